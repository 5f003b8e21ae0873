"""-m gpu: the abc-driven schedule (BQC_T_FLAG_ABC_DRIVEN) of the
CUDA path against the CPU oracle's abc-driven loop, per virtual triple and in total, and against the
library's own ijk-driven schedule.

Tolerance: the north_star one, |dE| <= 1e-10 |E| + 1e-12 Eh; per virtual triple
|de| <= 1e-10 |e_abc| + 1e-12 |E| / N.
"""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2502_17963_b200 as bqc
from bqc_inputs import make_config, make_inputs, worked_example
from gpu_util import dims, e_tol, to_device
from oracle import t_oracle as orc

pytestmark = pytest.mark.gpu

ABC = bqc.BQC_T_FLAG_ABC_DRIVEN

CASES = {
    "worked234": lambda: worked_example(2, 3, 4),
    "worked346": lambda: worked_example(3, 4, 6),
    "config1": lambda: make_config(1),
    "config1_t1": lambda: make_config(1, t1_std=0.05),
    "o8": lambda: make_inputs(8, 5, 10, seed=41, t1_std=0.05),     # exactly one 8-block of dual virtuals
    "o9": lambda: make_inputs(9, 6, 11, seed=42, t1_std=0.05),     # ragged dual tail
    "o17_v33": lambda: make_inputs(17, 33, 29, seed=43, t1_std=0.05),
    "v1": lambda: make_inputs(4, 1, 5, seed=44, t1_std=0.05),      # one virtual: no triples at all
    "o1": lambda: make_inputs(1, 6, 5, seed=45, t1_std=0.05),      # one occupied: E(T) = 0
}


def _run(inp, **kw):
    d = to_device(inp)
    o, v, X = dims(inp)
    f = kw.pop("f_ov", None)
    opts = bqc.make_opts(flags=ABC | kw.pop("flags", 0), f_ov=f, **kw)
    e_abc = torch.zeros(bqc.bqc_t_num_triplets(v), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(o, v, X, *d, opts=opts, e_triplet=e_abc)
    return e, e_abc.cpu().numpy()


@pytest.mark.parametrize("case", list(CASES))
def test_abc_driven_energy_and_per_virtual_triple_values(case):
    inp = CASES[case]()
    e, e_abc = _run(inp)
    e_ref, ref = orc.t_energy_abc(inp, return_triples=True)
    assert abs(e - e_ref) <= e_tol(e_ref)
    # per triple: relative part + the north_star absolute floor (1e-12 Eh) shared out over the triples
    tol = 1e-10 * np.abs(ref) + 1e-12 * max(abs(e_ref), 1.0) / max(len(ref), 1)
    assert np.all(np.abs(e_abc - ref) <= tol), np.max(np.abs(e_abc - ref) / tol)
    # diagonal virtual triples are skipped by the scheduler: exactly zero
    v = inp.nvir
    for a in range(v):
        assert e_abc[bqc.bqc_t_triplet_index(v, a, a, a)] == 0.0


def test_abc_and_ijk_schedules_agree_and_are_deterministic():
    inp = make_config(2, t1_std=0.05)
    d = to_device(inp)
    e_ijk = bqc.bqc_t_energy_ex(*dims(inp), *d)
    e1, t1 = _run(inp)
    e2, t2 = _run(inp)
    assert e1 == e2 and np.array_equal(t1, t2)            # bit-identical run to run
    assert abs(e1 - e_ijk) <= e_tol(e_ijk)
    # sampled virtual triples against the oracle (config 2: 76 virtuals, 20^3 tensors each)
    v = inp.nvir
    for (a, b, c) in [(0, 1, 2), (0, 0, v - 1), (3, v - 1, v - 1), (10, 40, 75), (v - 3, v - 2, v - 1)]:
        ref = orc.e_virtual_triple(inp, a, b, c)
        got = t1[bqc.bqc_t_triplet_index(v, a, b, c)]
        assert abs(got - ref) <= 1e-10 * abs(ref) + 1e-12 * abs(e_ijk) / len(t1)


def test_abc_driven_fock_term():
    rng = np.random.default_rng(23)
    base = make_inputs(5, 11, 14, seed=46, t1_std=0.05)
    inp = dataclasses.replace(base, f_ov=0.05 * rng.standard_normal((5, 11)))
    f = torch.from_numpy(inp.f_ov).cuda()
    e, e_abc = _run(inp, f_ov=f)
    e_ref, ref = orc.t_energy_abc(inp, return_triples=True)
    assert abs(e - e_ref) <= e_tol(e_ref)
    assert abs(e_ref - orc.t_energy_abc(base)) > 1e3 * e_tol(e_ref)      # the term carries weight
    np.testing.assert_allclose(e_abc, ref, rtol=1e-10, atol=1e-12 * abs(e_ref) / len(ref))


def test_abc_driven_windows_blocks_and_shards_are_bitwise_consistent():
    inp = make_inputs(6, 21, 17, seed=47, t1_std=0.05)
    v = inp.nvir
    e_all, t_all = _run(inp)
    # different virtual block sizes / batch sizes: same per-triple bits
    for kw in [dict(occ_block=4), dict(occ_block=7, max_batch=3), dict(max_batch=1)]:
        e, t = _run(inp, **kw)
        assert np.array_equal(t, t_all)
    # shards over virtual triples are disjoint and add up
    parts = [_run(inp, shard_rank=r, shard_count=3)[1] for r in range(3)]
    assert np.array_equal(sum(parts), t_all)
    for n in range(len(t_all)):
        assert sum(1 for p in parts if p[n] != 0.0) <= 1
    # whole block triples of virtuals per shard (BQC_T_FLAG_SHARD_BLOCKS): same bits, every triple once
    parts = [_run(inp, shard_rank=r, shard_count=4, occ_block=5, flags=bqc.BQC_T_FLAG_SHARD_BLOCKS)[1] for r in range(4)]
    assert np.array_equal(sum(parts), t_all)
    for n in range(len(t_all)):
        assert sum(1 for p in parts if p[n] != 0.0) <= 1
    # a virtual window [lo,hi): exactly the triples inside it
    lo, hi = 5, 14
    e_w, t_w = _run(inp, occ_lo=lo, occ_hi=hi)
    for a in range(v):
        for b in range(a, v):
            for c in range(b, v):
                n = bqc.bqc_t_triplet_index(v, a, b, c)
                inside = lo <= a and c < hi
                assert t_w[n] == (t_all[n] if inside else 0.0)
    opts = bqc.make_opts(flags=ABC, occ_lo=lo, occ_hi=hi)
    nwin = hi - lo
    ntrip = nwin * (nwin + 1) * (nwin + 2) // 6 - nwin
    assert bqc.bqc_t_flops(inp.nocc, v, opts) == ntrip * 12.0 * inp.nocc ** 3 * (v + inp.nocc)


def test_abc_driven_host_entry_point_and_workspace():
    inp = make_inputs(5, 12, 9, seed=48, t1_std=0.05)
    o, v, X = dims(inp)
    opts = bqc.make_opts(flags=ABC)
    host = [torch.from_numpy(np.ascontiguousarray(a)) for a in inp.arrays()]
    e_trip = torch.zeros(bqc.bqc_t_num_triplets(v), dtype=torch.float64)
    e, h2d, d2h = bqc.bqc_t_energy_host(o, v, X, *host, opts=opts, e_triplet=e_trip)
    e_ref, ref = orc.t_energy_abc(inp, return_triples=True)
    assert abs(e - e_ref) <= e_tol(e_ref)
    np.testing.assert_allclose(e_trip.numpy(), ref, rtol=1e-10, atol=1e-12 * abs(e_ref) / len(ref))
    assert d2h == 8 + 8 * len(ref)
    # caller workspace: exact size accepted, one byte less refused
    need = bqc.bqc_t_workspace_bytes(o, v, X, opts)
    d = to_device(inp)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    assert bqc.bqc_t_energy_ex(o, v, X, *d, opts=opts, workspace=ws) == e
    with pytest.raises(bqc.BqcError):
        bqc.bqc_t_energy_ex(o, v, X, *d, opts=opts, workspace=ws[: need - 1024])
