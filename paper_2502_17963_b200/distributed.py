"""One process per GPU: triplet sharding + the path's single exchange.

Triplets are independent, so each rank evaluates its share of them (`bqc_t_opts.shard_rank /
shard_count`; by default whole block triples, `BQC_T_FLAG_SHARD_BLOCKS`, so that a rank forms only the
(vv|ov) slabs its own triplets need) on its own replica of the inputs and there is no data-path
collective.  The only exchange is the final scalar: the per-rank partial sums are all-gathered and
added in rank order by the library (`bqc_sum_in_order`), so every rank returns the same bits and the
result does not depend on arrival order (an 8-byte all-reduce would do when that is not required).  Argument marshalling and
`torch.distributed` plumbing only — every step of the (T) path runs in the CUDA library.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

from . import binding as _b


def combine_partials(e_local: float, group=None, device=None) -> float:
    """All-gather the per-rank partial energies and add them in rank order (deterministic)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(e_local)
    world = dist.get_world_size(group)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else "cpu"
    mine = torch.tensor([e_local], dtype=torch.float64, device=device)
    parts = torch.zeros(world, dtype=torch.float64, device=device)
    dist.all_gather_into_tensor(parts, mine, group=group)
    return _b.bqc_sum_in_order(parts)      # the library's fixed-order sum: rank 0, 1, ... left to right


def bqc_t_energy_sharded(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, group=None,
                         flags=0, f_ov=None, occ_block=0, workspace=None, e_triplet=None) -> float:
    """E(T) over all ranks of `group`: this rank's shard through `bqc_t_energy_ex`, then `combine_partials`.

    Inputs are this rank's replicas (float64 CUDA tensors on the current device).  `e_triplet`, if given,
    receives this rank's per-triplet values (zeros elsewhere); summing it over ranks gives the full array.
    """
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    opts = _b.make_opts(occ_block=occ_block, shard_rank=rank, shard_count=world,
                        flags=flags | _b.BQC_T_FLAG_SHARD_BLOCKS, f_ov=f_ov)
    e_local = _b.bqc_t_energy_ex(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, opts=opts,
                                 workspace=workspace, e_triplet=e_triplet)
    return combine_partials(e_local, group)
