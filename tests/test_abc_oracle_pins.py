"""Pins of the oracle's abc-driven functions, -m "not gpu".

`oracle.t_oracle.w_virtual_triple / v_virtual_triple / e_virtual_triple / t_energy_abc` are pinned
against things other than themselves:
  * the dense six-index brute force of test_oracle_pins (W, V element by element; per-virtual-triple
    sums rebuilt from the six-index tensors),
  * the golden worked examples (totals printed in SURVEY.md §8(c) P2),
  * the first-principles Fock-space energy (no index formula),
  * the particle-hole duality of Eq. (2): exchanging the roles of occupied and virtual orbitals
    (with t2 -> -t2^T, eps -> -eps swapped, B_oo <-> B_vv) leaves E(T) unchanged and maps occupied
    triplets onto virtual triples.  The CUDA library's abc-driven schedule is built on this identity
    (with its own device-side transposes), so the identity itself is checked here on the CPU.
"""
import dataclasses
import itertools

import numpy as np
import pytest

from bqc_inputs import make_inputs, worked_example
from oracle import t_oracle as orc
from test_oracle_pins import _brute_force


def dual_inputs(inp):
    """The particle-hole dual problem (test helper; holds no (T) arithmetic)."""
    f = getattr(inp, "f_ov", None)
    return dataclasses.replace(
        inp, nocc=inp.nvir, nvir=inp.nocc,
        eps_occ=np.ascontiguousarray(-inp.eps_vir), eps_vir=np.ascontiguousarray(-inp.eps_occ),
        t1=np.ascontiguousarray(inp.t1.T),
        t2=np.ascontiguousarray(-inp.t2.transpose(2, 3, 0, 1)),
        B_oo=inp.B_vv.copy(), B_vv=inp.B_oo.copy(),
        B_ov=np.ascontiguousarray(inp.B_ov.transpose(0, 2, 1)),
        f_ov=None if f is None else np.ascontiguousarray(-f.T))


@pytest.fixture(scope="module")
def small():
    return make_inputs(4, 5, 9, seed=3, t1_std=0.05, t2_std=0.03)


def test_w_and_v_of_a_virtual_triple_match_the_six_index_brute_force(small):
    _, _, W6, V6 = _brute_force(small)
    for (a, b, c) in [(0, 1, 2), (1, 1, 3), (0, 2, 2), (4, 4, 4), (3, 0, 1)]:
        W = orc.w_virtual_triple(small, a, b, c)
        np.testing.assert_allclose(W, W6[:, :, :, a, b, c], rtol=1e-12, atol=1e-16)
        np.testing.assert_allclose(orc.v_virtual_triple(small, a, b, c, W), V6[:, :, :, a, b, c],
                                   rtol=1e-12, atol=1e-16)


def test_per_virtual_triple_values_from_the_six_index_tensors(small):
    """e_abc = (1/3) * sum over the distinct orderings of (a,b,c) of g_v, with
    g_v(a,b,c) = sum_ijk R V / D taken from the dense tensors (R permutes abc there)."""
    _, _, W, V = _brute_force(small)
    R = 4 * W + W.transpose(0, 1, 2, 4, 5, 3) + W.transpose(0, 1, 2, 5, 3, 4) \
        - 2 * (W.transpose(0, 1, 2, 3, 5, 4) + W.transpose(0, 1, 2, 5, 4, 3) + W.transpose(0, 1, 2, 4, 3, 5))
    eo, ev = small.eps_occ, small.eps_vir
    D = (eo[:, None, None, None, None, None] + eo[None, :, None, None, None, None]
         + eo[None, None, :, None, None, None] - ev[None, None, None, :, None, None]
         - ev[None, None, None, None, :, None] - ev[None, None, None, None, None, :])
    gv = (R * V / D).sum(axis=(0, 1, 2))
    total, e_abc = orc.t_energy_abc(small, return_triples=True)
    for n, (a, b, c) in enumerate(orc.triplet_list(small.nvir)):
        want = sum(gv[p] for p in set(itertools.permutations((a, b, c)))) / 3.0
        assert e_abc[n] == pytest.approx(want, rel=1e-11, abs=1e-18)
    assert total == pytest.approx(gv.sum() / 3.0, rel=1e-12)


def test_abc_driven_total_equals_the_golden_worked_examples():
    # E(T) of the closed-form inputs
    for shape, val in [((2, 3, 4), -9.406698159242249e-07), ((3, 4, 6), -1.851157457841839e-04)]:
        assert orc.t_energy_abc(worked_example(*shape)) == pytest.approx(val, rel=2e-12)


def test_abc_driven_total_equals_first_principles():
    from fock_space import first_principles_t
    inp = make_inputs(2, 3, 4, seed=5, t1_std=0.05, t2_std=0.05, f_std=0.1)
    e4, e5, ef = first_principles_t(inp, with_fock=True)
    assert orc.t_energy_abc(inp) == pytest.approx(e4 + e5 + ef, rel=1e-10)
    assert orc.t_energy_abc(inp, with_t1=False) == pytest.approx(e4, rel=1e-10)


def test_diagonal_virtual_triples_vanish(small):
    for a in range(small.nvir):
        assert abs(orc.e_virtual_triple(small, a, a, a)) < 1e-18


@pytest.mark.parametrize("fock", [False, True])
def test_particle_hole_duality(small, fock):
    inp = small
    if fock:
        rng = np.random.default_rng(17)
        inp = dataclasses.replace(small, f_ov=0.05 * rng.standard_normal((small.nocc, small.nvir)))
    d = dual_inputs(inp)
    e, e_ijk = orc.t_energy(inp, return_triplets=True)
    ed, e_dual = orc.t_energy(d, return_triplets=True)
    assert ed == pytest.approx(e, rel=1e-12)
    # the dual problem's occupied triplets are the virtual triples of the original one
    _, e_abc = orc.t_energy_abc(inp, return_triples=True)
    np.testing.assert_allclose(e_dual, e_abc, rtol=1e-11, atol=1e-18)
    # and twice dual is the identity
    dd = dual_inputs(d)
    for x, y in zip(dd.arrays(), inp.arrays()):
        np.testing.assert_array_equal(x, y)
    _, e_back = orc.t_energy_abc(d, return_triples=True)
    np.testing.assert_allclose(e_back, e_ijk, rtol=1e-11, atol=1e-18)
