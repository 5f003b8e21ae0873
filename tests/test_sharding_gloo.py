"""Multi-GPU path on CPU (gloo, world_size 2): the triplet sharding + the one exchange step.

Each rank takes the triplets the library assigns to it (bqc_t_triplet_owner — host logic of
libbqc_t.so), evaluates their e_ijk with the oracle standing in for the kernels (there is no GPU
here), and the per-triplet arrays are all-reduced exactly as bench.py / the binding do for N GPUs.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2502_17963_b200 as bqc
    from bqc_inputs import make_inputs
    from oracle import t_oracle as orc
    inp = make_inputs(4, 6, 9, seed=21, t1_std=0.05, t2_std=0.03)
    o = inp.nocc
    e = torch.zeros(bqc.bqc_t_num_triplets(o), dtype=torch.float64)
    mine = 0
    for (i, j, k) in orc.triplet_list(o):
        if bqc.bqc_t_triplet_owner(o, world, i, j, k) == rank:
            e[bqc.bqc_t_triplet_index(o, i, j, k)] = orc.e_triplet(inp, i, j, k)
            mine += 1
    # the library's own exchange step (paper_2502_17963_b200/distributed.py): all-gather + rank-order sum
    from paper_2502_17963_b200.distributed import combine_partials
    combined = combine_partials(float(e.sum()))
    ret[f"combined{rank}"] = combined
    dist.all_reduce(e, op=dist.ReduceOp.SUM)      # disjoint supports: the sum is exact
    total = float(e.sum())
    if rank == 0:
        ret["total"] = total
        ret["ref"] = orc.t_energy(inp)
    ret[f"count{rank}"] = mine
    dist.destroy_process_group()


def test_two_rank_sharded_energy_matches_single():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert ret["total"] == pytest.approx(ret["ref"], rel=1e-13)
    assert ret["combined0"] == ret["combined1"]                      # same bits on every rank
    assert ret["combined0"] == pytest.approx(ret["ref"], rel=1e-13)
    assert ret["count0"] + ret["count1"] == 20 and abs(ret["count0"] - ret["count1"]) <= 1
