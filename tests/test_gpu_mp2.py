"""-m gpu: the CUDA DF-MP2 path (Eq. (1)) against oracle/mp2_oracle.py.

Tolerance: |dE| <= 1e-10 |E| + 1e-12 Eh (the north_star bar); per pair
|de_ij| <= 1e-10 |e_ij| + 1e-12 |E| / o^2.  Both sides are FP64; each (ia|jb) is a sum of naux products in a
different order than BLAS (relative error ~ sqrt(naux) 2^-53), far below the bar.
"""
import numpy as np
import pytest
import torch

import paper_2502_17963_b200 as bqc
from bqc_inputs import make_config, make_inputs
from oracle import mp2_oracle as mp2

pytestmark = pytest.mark.gpu


def _dev(inp):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (inp.eps_occ, inp.eps_vir, inp.B_ov)]


CASES = {
    "config1": lambda: make_config(1),
    "config2": lambda: make_config(2),
    "tiny": lambda: make_inputs(1, 1, 1, seed=3),
    "ragged": lambda: make_inputs(7, 33, 29, seed=4),          # v = one tile + 1, odd naux
    "ragged2": lambda: make_inputs(3, 65, 50, seed=6),         # three tiles, ragged tail of one
    "wide": lambda: make_inputs(2, 131, 17, seed=9),           # 5 x 5 tile pairs, K tail
}


@pytest.mark.parametrize("case", sorted(CASES))
def test_mp2_energy_and_pairs(case):
    inp = CASES[case]()
    o, v, X = inp.nocc, inp.nvir, inp.naux
    d = _dev(inp)
    e_ref = mp2.mp2_energy(inp)
    pairs_ref = mp2.pair_energies(inp)
    e_pair = torch.full((o, o), 7.0, dtype=torch.float64, device="cuda")
    e_gpu = bqc.bqc_mp2_energy_ex(o, v, X, *d, e_pair=e_pair)
    assert abs(e_gpu - e_ref) <= 1e-10 * abs(e_ref) + 1e-12
    got = e_pair.cpu().numpy()
    tol = 1e-10 * np.abs(pairs_ref) + 1e-12 * abs(e_ref) / (o * o)
    assert np.all(np.abs(got - pairs_ref) <= tol), np.max(np.abs(got - pairs_ref))
    assert np.array_equal(got, got.T)
    # the plain entry point
    assert bqc.bqc_mp2_energy(o, v, X, *d) == e_gpu


def test_mp2_blocking_and_sharding_are_bitwise_consistent():
    inp = make_inputs(9, 40, 37, seed=12)
    o, v, X = inp.nocc, inp.nvir, inp.naux
    d = _dev(inp)
    ref_pair = torch.zeros((o, o), dtype=torch.float64, device="cuda")
    e_ref = bqc.bqc_mp2_energy_ex(o, v, X, *d, opts=bqc.make_mp2_opts(occ_block=9), e_pair=ref_pair)
    assert bqc.bqc_mp2_energy_ex(o, v, X, *d, opts=bqc.make_mp2_opts(occ_block=9)) == e_ref    # run to run
    for bi in (1, 2, 4):
        p = torch.zeros((o, o), dtype=torch.float64, device="cuda")
        e = bqc.bqc_mp2_energy_ex(o, v, X, *d, opts=bqc.make_mp2_opts(occ_block=bi), e_pair=p)
        assert torch.equal(p, ref_pair)          # each e_ij is the same arithmetic whatever the blocking
        assert e == e_ref
    # two shards: disjoint rows, pair matrices add up bit-exactly, energies add up to rounding
    parts, es = [], []
    for r in range(2):
        p = torch.zeros((o, o), dtype=torch.float64, device="cuda")
        es.append(bqc.bqc_mp2_energy_ex(o, v, X, *d, opts=bqc.make_mp2_opts(occ_block=2, shard_rank=r, shard_count=2),
                                        e_pair=p))
        parts.append(p)
    assert torch.equal(torch.triu(parts[0]) + torch.triu(parts[1]), torch.triu(ref_pair))
    assert abs(es[0] + es[1] - e_ref) <= 1e-13 * abs(e_ref)


def test_mp2_host_entry_point_and_errors():
    inp = make_inputs(4, 21, 13, seed=2)
    o, v, X = inp.nocc, inp.nvir, inp.naux
    host = [torch.from_numpy(np.ascontiguousarray(a)) for a in (inp.eps_occ, inp.eps_vir, inp.B_ov)]
    pair = torch.zeros((o, o), dtype=torch.float64)
    e, h2d, d2h = bqc.bqc_mp2_energy_host(o, v, X, *host, e_pair=pair)
    assert h2d == 8 * (o + v + X * o * v) and d2h == 8 + 8 * o * o
    e_ref = mp2.mp2_energy(inp)
    assert abs(e - e_ref) <= 1e-10 * abs(e_ref) + 1e-12
    np.testing.assert_allclose(pair.numpy(), mp2.pair_energies(inp), rtol=1e-10, atol=1e-14)
    d = _dev(inp)
    bad = d[0].clone()
    bad[-1] = 5.0                                    # occupied level above the lowest virtual
    with pytest.raises(bqc.BqcError) as ei:
        bqc.bqc_mp2_energy_ex(o, v, X, bad, d[1], d[2])
    assert ei.value.code == 8                        # BQC_ERR_DENOMINATOR
    with pytest.raises(bqc.BqcError):
        bqc.bqc_mp2_energy_ex(o, v, X, *d, opts=bqc.make_mp2_opts(shard_rank=3, shard_count=2))
    # caller workspace: same bits as the internally allocated one; too small is refused
    e_dev = bqc.bqc_mp2_energy_ex(o, v, X, *d)
    need = bqc.bqc_mp2_workspace_bytes(o, v, X)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    assert bqc.bqc_mp2_energy_ex(o, v, X, *d, opts=bqc.make_mp2_opts(workspace=ws)) == e_dev == e
    with pytest.raises(bqc.BqcError) as ei:
        bqc.bqc_mp2_energy_ex(o, v, X, *d, opts=bqc.make_mp2_opts(workspace=ws[: need - 1024]))
    assert ei.value.code == 5                        # BQC_ERR_WORKSPACE


def test_mp2_config3_sampled_pairs():
    """BASELINE.json configs[2] shape (o=40, v=152, X=672): full energy plus sampled pairs against the oracle."""
    inp = make_config(3)
    o, v, X = inp.nocc, inp.nvir, inp.naux
    d = _dev(inp)
    e_pair = torch.zeros((o, o), dtype=torch.float64, device="cuda")
    e_gpu = bqc.bqc_mp2_energy_ex(o, v, X, *d, e_pair=e_pair)
    got = e_pair.cpu().numpy()
    rng = np.random.default_rng(33)
    pairs = [(0, 0), (o - 1, o - 1), (0, o - 1), (17, 18)] + [tuple(sorted(rng.integers(0, o, 2))) for _ in range(12)]
    for (i, j) in pairs:
        ref = mp2.pair_energy(inp, i, j)
        assert abs(got[i, j] - ref) <= 1e-10 * abs(ref) + 1e-12 * abs(e_gpu) / (o * o)
        assert got[j, i] == got[i, j]
    tri = sum((2 - (i == j)) * got[i, j] for i in range(o) for j in range(i, o))
    assert abs(tri - e_gpu) <= 1e-12 * abs(e_gpu)
    e_ref = mp2.mp2_energy(inp)
    assert abs(e_gpu - e_ref) <= 1e-10 * abs(e_ref) + 1e-12
