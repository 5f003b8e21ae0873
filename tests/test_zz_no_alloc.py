"""-m gpu: bqc_sum_fixed_noalloc — the library's one entry point that allocates nothing (include/bqc_t.h).

Its scratch lives in a file-scope `static __device__` array (32 KiB per GPU), so callers that cannot call
cudaMalloc (CUDA-graph capture, tight serving loops) can still take the fixed-order final sum of the (T) path.
The output is checked against the existing paths — the E(T) that bqc_t_energy_ex returns for the same e_ijk array
(final_sum_kernel) and bqc_sum_in_order — within the north_star tolerance, on two calls in a row that share the
scratch array (the second one shorter, so stale partial sums of the first sit behind the slots it uses).

This file is named to be collected LAST (the suite runs with pytest -x).  It passes alone in a fresh process
(the scratch address is looked up on first use) and after the other tests.
"""
import numpy as np
import pytest
import torch

import paper_2502_17963_b200 as bqc
from bqc_inputs import make_inputs
from gpu_util import dims, e_tol, to_device

pytestmark = pytest.mark.gpu


def test_no_alloc_sum_matches_the_existing_paths_on_two_calls_in_a_row():
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")

    # call 1: a long array of same-sign values (the shape of an e_ijk array: all <= 0), several hundred chunks + a ragged tail
    rng = np.random.default_rng(314)
    n1 = 1_234_567
    x1 = torch.from_numpy(-rng.random(n1) * 10.0 ** rng.integers(-6, 1, n1)).cuda()
    bqc.bqc_sum_fixed_noalloc(x1, out)
    s1 = float(out.item())
    ref1 = bqc.bqc_sum_in_order(x1)                       # existing path: strictly sequential sum on the device
    assert abs(s1 - ref1) <= e_tol(ref1)
    assert abs(s1 - float(x1.sum().item())) <= e_tol(ref1)

    # call 2, right after, shorter (2 chunks): the per-triplet energies of a real evaluation; the existing path's
    # own final sum (final_sum_kernel inside bqc_t_energy_ex) is the reference.  Stale slots of call 1 must not leak.
    inp = make_inputs(7, 21, 30, seed=77, t1_std=0.05, t2_std=0.03)
    d = to_device(inp)
    et = torch.empty(bqc.bqc_t_num_triplets(inp.nocc), dtype=torch.float64, device="cuda")
    e = bqc.bqc_t_energy_ex(*dims(inp), *d, e_triplet=et)
    x2 = et.repeat(60)                                    # 5 040 elements: one full chunk + a tail
    out.fill_(float("nan"))
    bqc.bqc_sum_fixed_noalloc(x2, out)
    s2 = float(out.item())
    assert abs(s2 - 60.0 * e) <= e_tol(60.0 * e)
    assert abs(s2 - bqc.bqc_sum_in_order(x2)) <= e_tol(60.0 * e)

    # same input twice -> same bits (fixed order, shared scratch fully rewritten)
    out2 = torch.empty_like(out)
    bqc.bqc_sum_fixed_noalloc(x1, out2)
    assert float(out2.item()) == s1
    bqc.bqc_sum_fixed_noalloc(x2, out2)
    assert float(out2.item()) == s2

    # edge cases: empty input, one element, exactly one chunk
    bqc.bqc_sum_fixed_noalloc(x1[:0], out)
    assert float(out.item()) == 0.0
    bqc.bqc_sum_fixed_noalloc(x1[:1], out)
    assert float(out.item()) == float(x1[0].item())
    bqc.bqc_sum_fixed_noalloc(x1[:4096], out)
    assert abs(float(out.item()) - bqc.bqc_sum_in_order(x1[:4096])) <= e_tol(float(out.item()))


def test_no_alloc_sum_rejects_sizes_beyond_the_static_scratch():
    nmax = bqc.bqc_sum_fixed_noalloc_max()
    assert nmax == 4096 * 4096
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    x = torch.zeros(nmax + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(bqc.BqcError) as ei:
        bqc.bqc_sum_fixed_noalloc(x, out)
    assert ei.value.code == 1 and "exceeds the maximum" in str(ei.value)
    bqc.bqc_sum_fixed_noalloc(x[:nmax], out)              # the maximum itself is accepted
    assert float(out.item()) == 0.0
    # host pointers are refused, not dereferenced
    with pytest.raises(ValueError):
        bqc.bqc_sum_fixed_noalloc(torch.zeros(4, dtype=torch.float64), out)
