"""SURVEY.md §8(e) sharding on CPU: world_size-2 gloo run of the partition + the one collective (all-gather of the owned
displacement slabs).  The local assembler of this test is the oracle (no GPU here): every rank's owned rows, residual and
pattern must equal the corresponding rows of the global assembly bit for bit (same summation order by construction)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _check_rank(cfg, world, rank, group_ok=True):
    import oracle
    from paper_2606_17390_b200 import shard
    coords, conn, u = cfg["coords"], cfg["conn"], cfg["u"]
    nn, ne = coords.shape[0], conn.shape[0]
    gmat = oracle.mat_from_desc(cfg["matdesc"], ne)
    rp, ci, _ = oracle.pattern(nn, conn, with_slots=False)
    g = oracle.assemble(coords, conn, u, cfg["hist_in"], gmat, rp, ci)
    p = shard.partition(nn, conn, world, rank)
    u_owned = torch.from_numpy(u[p["n0"]:p["n1"]].ravel().copy())
    u_local = shard.exchange_u(u_owned, p).numpy().reshape(-1, 3)
    assert np.array_equal(u_local, u[p["lnodes"]])                       # ghost values arrived through the collective
    lcoords = coords[p["lnodes"]]
    lmat = gmat if gmat.shape[0] == 1 else gmat[p["elems"]]
    lrp, lci, _ = oracle.pattern(lcoords.shape[0], p["lconn"], with_slots=False)
    o = oracle.assemble(lcoords, p["lconn"], u_local, cfg["hist_in"][p["elems"]], lmat, lrp, lci)
    a, b = lrp[3 * p["lo"]], lrp[3 * p["hi"]]
    ga, gb = rp[3 * p["n0"]], rp[3 * p["n1"]]
    assert b - a == gb - ga
    assert np.array_equal(lrp[3 * p["lo"]:3 * p["hi"] + 1] - a, rp[3 * p["n0"]:3 * p["n1"] + 1] - ga)
    lcol = lci[a:b].astype(np.int64)
    assert np.array_equal(3 * p["lnodes"][lcol // 3] + lcol % 3, ci[ga:gb])     # global column ids, same order
    assert np.array_equal(o["csr_vals"][a:b], g["csr_vals"][ga:gb])             # bit for bit
    assert np.array_equal(o["residual"][3 * p["lo"]:3 * p["hi"]], g["residual"][3 * p["n0"]:3 * p["n1"]])
    assert np.array_equal(o["hist_out"], g["hist_out"][p["elems"]])
    return int(p["elems"].size), ne


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import synth
    res = []
    for cfg in (synth.make_config(3, n=6), synth.make_config(4, n=8)):
        res.append(_check_rank(cfg, world, rank))
    out[rank] = res
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_reproduces_the_global_rows():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29531, out), nprocs=2, join=True)
    for k in range(2):
        (e0, ne), (e1, _) = out[0][k], out[1][k]
        assert e0 + e1 >= ne and e0 < ne and e1 < ne          # every element somewhere, ghost layer recomputed, no full copy


def test_partition_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import synth
    from paper_2606_17390_b200 import shard
    cfg = synth.make_config(4, n=6)
    p = shard.partition(cfg["coords"].shape[0], cfg["conn"], 1, 0)
    assert np.array_equal(p["elems"], np.arange(cfg["conn"].shape[0])) and np.array_equal(p["lconn"], cfg["conn"])
    assert (p["lo"], p["hi"]) == (0, cfg["coords"].shape[0])
