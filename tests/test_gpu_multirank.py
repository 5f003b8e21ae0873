"""-m gpu: two ranks through the REAL library.

One process per rank, world_size 2, gloo backend, both ranks on cuda:0 — their kernels never wait on one
another (triplets are independent; the only exchange is a host-side scalar), so sharing the one GPU of
the test box is safe.  `bqc_t_energy_sharded` deals whole block triples (BQC_T_FLAG_SHARD_BLOCKS); the
combined energy and the sum of the per-rank per-triplet arrays are compared with the oracle.
Also: bench.py --gpus 2 starts its own ranks, and refuses to when fewer than 2 GPUs are visible.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, ret, abc):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    import paper_2502_17963_b200 as bqc
    from bqc_inputs import make_inputs
    inp = make_inputs(7, 21, 30, seed=77, t1_std=0.05, t2_std=0.03)
    o, v, X = inp.nocc, inp.nvir, inp.naux
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in inp.arrays()]
    nidx = v if abc else o
    e_trip = torch.zeros(bqc.bqc_t_num_triplets(nidx), dtype=torch.float64, device="cuda")
    flags = bqc.BQC_T_FLAG_ABC_DRIVEN if abc else 0
    bo = 5 if abc else 2
    e = bqc.bqc_t_energy_sharded(o, v, X, *dev, flags=flags, occ_block=bo, e_triplet=e_trip)
    ret[f"e{rank}"] = e
    ret[f"trip{rank}"] = e_trip.cpu().numpy()
    # what this rank should have evaluated according to the host-side owner map
    opts = bqc.make_opts(occ_block=bo, shard_count=world, flags=flags | bqc.BQC_T_FLAG_SHARD_BLOCKS)
    own = np.zeros(e_trip.numel(), dtype=bool)
    for i in range(nidx):
        for j in range(i, nidx):
            for k in range(j, nidx):
                if bqc.bqc_t_triplet_owner_ex(o, v, X, opts, i, j, k) == rank and not (i == j == k):
                    own[bqc.bqc_t_triplet_index(nidx, i, j, k)] = True
    ret[f"own{rank}"] = own
    dist.destroy_process_group()


@pytest.mark.parametrize("abc", [False, True])
def test_two_ranks_through_the_cuda_library(abc):
    from bqc_inputs import make_inputs
    from oracle import t_oracle as orc
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(2, port, ret, abc), nprocs=2, join=True)
    inp = make_inputs(7, 21, 30, seed=77, t1_std=0.05, t2_std=0.03)
    e_ref = orc.t_energy(inp)
    tol = 1e-10 * abs(e_ref) + 1e-12
    assert ret["e0"] == ret["e1"]                                   # every rank returns the same bits
    assert abs(ret["e0"] - e_ref) <= tol
    t0, t1 = ret["trip0"], ret["trip1"]
    own0, own1 = ret["own0"], ret["own1"]
    assert not (own0 & own1).any()                                  # shards are disjoint ...
    assert not t0[~own0].any() and not t1[~own1].any()              # ... each rank wrote only its own triplets
    total = t0 + t1
    if abc:
        n = inp.nvir
        ref = np.array([orc.e_virtual_triple(inp, a, b, c) for a in range(n) for b in range(a, n) for c in range(b, n)])
    else:
        n = inp.nocc
        ref = np.array([orc.e_triplet(inp, i, j, k) for (i, j, k) in orc.triplet_list(n)])
    assert np.all(np.abs(total - ref) <= 1e-10 * np.abs(ref) + 1e-12 * abs(e_ref) / len(ref))
    assert abs(total.sum() - e_ref) <= tol


def _bench(*argv):
    env = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], capture_output=True, text=True,
                          env=env, timeout=900)


def test_bench_starts_its_own_ranks():
    """bench.py --gpus 2 (no torchrun): two ranks, strong scaling over block triples, n_gpus = 2.  On a 1-GPU
    box the ranks share cuda:0 (--share-gpu, test mode: the timings mean nothing, the plumbing is what runs)."""
    share = [] if torch.cuda.device_count() >= 2 else ["--share-gpu"]
    r = _bench("--gpus", "2", "--config", "2", "--full", "--steps", "1", "--warmup", "1", "--e2e-steps", "1",
               "--peak-seconds", "0.2", "--occ-block", "5", *share)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                          # rank 0 prints ONE line
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["scaling"] == "strong"
    per = out["ranks"]["per_rank"]
    assert [p["rank"] for p in per] == [0, 1]
    assert sum(p["triplets"] for p in per) == 1540 - 20             # config 2: every non-diagonal triplet once
    assert out["ranks"]["load_imbalance_max_over_mean_flops"] < 1.2
    # the combined energy equals the single-rank full evaluation to rounding
    r1 = _bench("--gpus", "1", "--config", "2", "--full", "--steps", "1", "--warmup", "1", "--e2e-steps", "0",
                "--peak-seconds", "0.2", "--no-cpu-baseline")
    assert r1.returncode == 0, r1.stderr[-2000:]
    e1 = json.loads([ln for ln in r1.stdout.splitlines() if ln.startswith("{")][0])["e_t_of_step_hartree"]
    assert abs(out["e_t_of_step_hartree"] - e1) <= 1e-12 * abs(e1)


def test_bench_refuses_more_ranks_than_gpus():
    n = torch.cuda.device_count()
    r = _bench("--gpus", str(n + 1), "--steps", "1", "--warmup", "1")
    assert r.returncode != 0
    assert "CUDA device(s) visible" in (r.stderr + r.stdout)
