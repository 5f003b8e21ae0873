"""Pins of oracle/mp2_oracle.py (Eq. (1)).  None re-types the
oracle's own expression: first principles (no index formula), a hand-computed closed form, the spin-component
decomposition on dense four-index tensors, scaling laws, relabelling, plain Python loops."""
import copy
import itertools

import numpy as np
import pytest

from bqc_inputs import make_inputs
from oracle import mp2_oracle as mp2
from fock_space import first_principles_mp2


@pytest.mark.parametrize("shape,seed", [((2, 2, 5), 7), ((3, 2, 4), 11), ((2, 3, 4), 5), ((1, 3, 3), 2)])
def test_mp2_matches_second_order_perturbation_theory(shape, seed):
    """E2 = <0|W_N R W_N|0> on the Fock space of 2(o+v) spin orbitals fixes the spin factors 2 / -1, the
    index pairing (ia|jb) vs (ib|ja), the sign of the denominator and the unrestricted i,j,a,b sum."""
    inp = make_inputs(*shape, seed=seed)
    e2_d, e2_s = first_principles_mp2(inp)
    assert abs(e2_s) < 1e-14 * abs(e2_d)          # Brillouin: no singles with a normal-ordered W_N
    assert e2_d < 0
    assert mp2.mp2_energy(inp) == pytest.approx(e2_d, rel=1e-11)


def test_closed_form_one_occupied_two_virtuals():
    """o=1, v=2, X=1 by hand: (ia|ib) = x_a x_b with x = B_ov[0,0,:];
    E = x0^4/(2(e-e0)) + x1^4/(2(e-e1)) + 2 x0^2 x1^2 /(2e-e0-e1)   (the a!=b terms: (2-1) x_a^2 x_b^2 each)."""
    inp = make_inputs(1, 2, 1, seed=3)
    x0, x1 = 0.3, -0.7
    inp.B_ov[0, 0, :] = (x0, x1)
    inp.eps_occ[:] = -0.5
    inp.eps_vir[:] = (0.25, 1.5)
    e, e0, e1 = -0.5, 0.25, 1.5
    want = x0 ** 4 / (2 * (e - e0)) + x1 ** 4 / (2 * (e - e1)) + 2 * x0 ** 2 * x1 ** 2 / (2 * e - e0 - e1)
    assert mp2.mp2_energy(inp) == pytest.approx(want, rel=1e-14)
    assert mp2.pair_energy(inp, 0, 0) == pytest.approx(want, rel=1e-14)


def _dense(inp):
    ovov = np.einsum("Qia,Qjb->iajb", inp.B_ov, inp.B_ov)
    eo, ev = inp.eps_occ, inp.eps_vir
    D = eo[:, None, None, None] + eo[None, None, :, None] - ev[None, :, None, None] - ev[None, None, None, :]
    return ovov, D


def test_spin_component_decomposition_dense():
    """E = E_os + E_ss with E_os = sum (ia|jb)^2/D and E_ss = 1/2 sum [(ia|jb)-(ib|ja)]^2/D, both <= 0, on
    dense four-index tensors (one einsum, no pair loop)."""
    inp = make_inputs(4, 6, 9, seed=21)
    g, D = _dense(inp)
    e_os = np.sum(g * g / D)
    anti = g - g.transpose(0, 3, 2, 1)
    e_ss = 0.5 * np.sum(anti * anti / D)
    assert e_os < 0 and e_ss < 0
    assert mp2.mp2_energy(inp) == pytest.approx(e_os + e_ss, rel=1e-12)


def test_plain_loops_and_pair_symmetry():
    inp = make_inputs(3, 4, 5, seed=8)
    o, v, X = 3, 4, 5

    def integral(i, a, j, b):
        return sum(inp.B_ov[Q, i, a] * inp.B_ov[Q, j, b] for Q in range(X))

    tot = 0.0
    pair = np.zeros((o, o))
    for i, j, a, b in itertools.product(range(o), range(o), range(v), range(v)):
        t = integral(i, a, j, b) * (2 * integral(i, a, j, b) - integral(i, b, j, a)) / (
            inp.eps_occ[i] + inp.eps_occ[j] - inp.eps_vir[a] - inp.eps_vir[b])
        tot += t
        pair[i, j] += t
    e = mp2.pair_energies(inp)
    np.testing.assert_allclose(e, pair, rtol=1e-12, atol=0)
    np.testing.assert_allclose(e, e.T, rtol=1e-12, atol=0)                     # e_ij = e_ji
    assert mp2.mp2_energy(inp) == pytest.approx(tot, rel=1e-12)
    tri = sum((2 - (i == j)) * e[i, j] for i in range(o) for j in range(i, o))   # the i<=j form the GPU uses
    assert mp2.mp2_energy(inp) == pytest.approx(tri, rel=1e-13)


def test_scaling_laws_and_relabelling():
    inp = make_inputs(3, 5, 7, seed=13)
    e = mp2.mp2_energy(inp)
    s = copy.deepcopy(inp)
    s.B_ov = 1.7 * inp.B_ov
    assert mp2.mp2_energy(s) == pytest.approx(1.7 ** 4 * e, rel=1e-12)          # quartic in B
    s = copy.deepcopy(inp)
    s.eps_occ, s.eps_vir = 2.5 * inp.eps_occ, 2.5 * inp.eps_vir
    assert mp2.mp2_energy(s) == pytest.approx(e / 2.5, rel=1e-12)               # 1/eps
    s = copy.deepcopy(inp)                                                      # uniform shift cancels in D
    s.eps_occ, s.eps_vir = inp.eps_occ + 0.3, inp.eps_vir + 0.3
    assert mp2.mp2_energy(s) == pytest.approx(e, rel=1e-12)
    po, pv = np.array([2, 0, 1]), np.array([4, 2, 0, 1, 3])
    s = copy.deepcopy(inp)
    s.B_ov = np.ascontiguousarray(inp.B_ov[:, po][:, :, pv])
    s.eps_occ, s.eps_vir = inp.eps_occ[po], inp.eps_vir[pv]
    assert mp2.mp2_energy(s) == pytest.approx(e, rel=1e-12)
    # a sign flip of one auxiliary vector leaves every (ia|jb) unchanged
    s = copy.deepcopy(inp)
    s.B_ov[2] *= -1.0
    assert mp2.mp2_energy(s) == pytest.approx(e, rel=1e-13)


def test_a_wrong_exchange_pairing_or_factor_would_be_caught():
    """The pins above must move if the exchange integral were (ia|jb) itself, (ja|ib)-transposed wrongly, or
    the factor 2 dropped: check the three wrong variants differ from the dense truth at the 1e-3 level."""
    inp = make_inputs(3, 4, 6, seed=5)
    g, D = _dense(inp)
    truth = np.sum(g * (2 * g - g.transpose(0, 3, 2, 1)) / D)
    wrong = [np.sum(g * (2 * g - g) / D), np.sum(g * (g - g.transpose(0, 3, 2, 1)) / D),
             np.sum(g * (2 * g + g.transpose(0, 3, 2, 1)) / D)]
    assert mp2.mp2_energy(inp) == pytest.approx(truth, rel=1e-12)
    for w in wrong:
        assert abs(w - truth) > 1e-3 * abs(truth)
