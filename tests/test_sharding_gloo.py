"""Multi-GPU path on CPU (gloo, world_size 2): the triplet sharding + the one exchange step.

Each rank takes the triplets the library assigns to it — by whole block triples
(BQC_T_FLAG_SHARD_BLOCKS, the split `bqc_t_energy_sharded` and `bench.py --full` use; host logic
`bqc_t_triplet_owner_ex`) and by the per-triplet modulo (`bqc_t_triplet_owner`) — evaluates their e_ijk
with the oracle standing in for the kernels (there is no GPU here), and the partial sums are combined by
the product's exchange step (`combine_partials`: all-gather + the library's `bqc_sum_in_order`).
The same two ranks through the real CUDA kernels: tests/test_gpu_multirank.py (-m gpu).
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
    from paper_2502_17963_b200.distributed import combine_partials
    inp = make_inputs(4, 6, 9, seed=21, t1_std=0.05, t2_std=0.03)
    o, v, X = inp.nocc, inp.nvir, inp.naux
    blocks = bqc.make_opts(occ_block=2, shard_count=world, flags=bqc.BQC_T_FLAG_SHARD_BLOCKS)
    for mode in ("blocks", "modulo"):
        e = torch.zeros(bqc.bqc_t_num_triplets(o), dtype=torch.float64)
        mine = 0
        for (i, j, k) in orc.triplet_list(o):
            owner = (bqc.bqc_t_triplet_owner_ex(o, v, X, blocks, i, j, k) if mode == "blocks"
                     else bqc.bqc_t_triplet_owner(o, world, i, j, k))
            assert 0 <= owner < world
            if owner == rank:
                e[bqc.bqc_t_triplet_index(o, i, j, k)] = orc.e_triplet(inp, i, j, k)
                mine += 1
        # the library's own exchange step (paper_2502_17963_b200/distributed.py)
        ret[f"{mode}.combined{rank}"] = combine_partials(float(e.sum()))
        ret[f"{mode}.partial{rank}"] = float(e.sum())
        dist.all_reduce(e, op=dist.ReduceOp.SUM)      # disjoint supports: the sum is exact
        ret[f"{mode}.total{rank}"] = float(e.sum())
        ret[f"{mode}.count{rank}"] = mine
    if rank == 0:
        ret["ref"] = orc.t_energy(inp)
        # the flop model deals the same triplets: per-rank share of bqc_t_flops
        ret["flops"] = [bqc.bqc_t_flops(o, v, bqc.make_opts(occ_block=2, shard_rank=r, shard_count=world,
                                                          flags=bqc.BQC_T_FLAG_SHARD_BLOCKS)) for r in range(world)]
    dist.destroy_process_group()


def test_two_rank_sharded_energy_matches_single():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    for mode in ("blocks", "modulo"):
        assert ret[f"{mode}.total0"] == pytest.approx(ret["ref"], rel=1e-13)
        assert ret[f"{mode}.combined0"] == ret[f"{mode}.combined1"]               # same bits on every rank
        assert ret[f"{mode}.combined0"] == ret[f"{mode}.partial0"] + ret[f"{mode}.partial1"]   # rank order
        assert ret[f"{mode}.combined0"] == pytest.approx(ret["ref"], rel=1e-13)
        assert ret[f"{mode}.count0"] + ret[f"{mode}.count1"] == 20
    assert abs(ret["modulo.count0"] - ret["modulo.count1"]) <= 1
    # block-triple split of 2 blocks of 2 orbitals: 4 block triples dealt round-robin; the non-diagonal
    # triplet counts the flop model reports are those of the owner map
    per = 12.0 * 6 ** 3 * (6 + 4)
    assert sum(ret["flops"]) == 16 * per                                          # 20 triplets - 4 diagonal


def test_sum_in_order_is_left_to_right():
    """bqc_sum_in_order on a host array: strictly sequential FP64 addition (no GPU needed)."""
    import paper_2502_17963_b200 as bqc
    x = torch.tensor([1.0, 1e-16, 1e-16, -1.0, 3e-17], dtype=torch.float64)
    s = 0.0
    for t in x.tolist():
        s += t
    assert bqc.bqc_sum_in_order(x) == s == 3e-17           # a pairwise tree would give 1e-16 + ... != this
    assert bqc.bqc_sum_in_order(torch.zeros(0, dtype=torch.float64)) == 0.0
    rng = np.random.default_rng(5)
    y = torch.from_numpy(rng.standard_normal(1000) * 10.0 ** rng.integers(-8, 8, 1000))
    s = 0.0
    for t in y.tolist():
        s += t
    assert bqc.bqc_sum_in_order(y) == s


def test_block_triple_owner_matches_the_flop_model():
    import paper_2502_17963_b200 as bqc
    F = bqc.BQC_T_FLAG_SHARD_BLOCKS
    for (o, v, bo, world) in [(7, 11, 2, 3), (20, 76, 0, 2), (9, 5, 4, 8)]:
        counts = [0] * world
        for i in range(o):
            for j in range(i, o):
                for k in range(j, o):
                    r = bqc.bqc_t_triplet_owner_ex(o, v, 10, bqc.make_opts(occ_block=bo, shard_count=world, flags=F),
                                                   i, j, k)
                    assert 0 <= r < world
                    if not (i == j == k):
                        counts[r] += 1
        for r in range(world):
            fl = bqc.bqc_t_flops(o, v, bqc.make_opts(occ_block=bo, shard_rank=r, shard_count=world, flags=F))
            assert fl == counts[r] * 12.0 * v ** 3 * (v + o)
    # outside the window / unordered -> -1
    assert bqc.bqc_t_triplet_owner_ex(7, 11, 10, bqc.make_opts(occ_lo=2, occ_hi=5, shard_count=2, flags=F), 0, 2, 3) == -1
    assert bqc.bqc_t_triplet_owner_ex(7, 11, 10, bqc.make_opts(shard_count=2), 3, 2, 4) == -1
