"""Pins of the CPU oracle (-m "not gpu"): golden worked examples, brute force,
alternative published forms, invariants and special cases."""
import copy
import itertools
import os

import numpy as np
import pytest

from bqc_inputs import make_inputs, make_config, worked_example, sample_triplets
from oracle import t_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")


def _gold():
    rows = []
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if line:
            f = line.split()
            rows.append((f[0], tuple(int(x) for x in f[1:4]),
                         tuple(int(x) for x in f[4:-1]), float(f[-1])))
    return rows


@pytest.fixture(scope="module")
def worked():
    return {s: worked_example(*s) for s in [(2, 3, 4), (3, 4, 6)]}


@pytest.mark.parametrize("row", _gold(), ids=lambda r: f"{r[0]}-{r[1]}-{r[2]}")
def test_golden_worked_examples(worked, row):
    kind, shape, key, val = row
    inp = worked[shape]
    if kind == "E4":
        got = orc.t_energy(inp, with_t1=False)
    elif kind == "E5":
        got = orc.t_energy(inp) - orc.t_energy(inp, with_t1=False)
    elif kind == "ET":
        got = orc.t_energy(inp)
    elif kind == "e":
        got = orc.e_triplet(inp, *key)
    elif kind == "eri":
        b, d, i, a = key
        got = orc.slab_vvov(inp, i)[a, b, d]
    elif kind in ("W", "V", "D"):
        i, j, k, a, b, c = key
        W = orc.w_triplet(inp, i, j, k)
        got = {"W": W, "V": orc.v_triplet(inp, i, j, k, W),
               "D": orc.d_triplet(inp, i, j, k)}[kind][a, b, c]
    if val == 0.0:
        assert abs(got) < 1e-20
    else:
        assert got == pytest.approx(val, rel=2e-12)


# ---- P4: brute force through the full six-index W -------------------------
def _full_mo(inp):
    o, n = inp.nocc, inp.nocc + inp.nvir
    B = np.zeros((inp.naux, n, n))
    B[:, :o, :o] = inp.B_oo
    B[:, :o, o:] = inp.B_ov
    B[:, o:, :o] = inp.B_ov.transpose(0, 2, 1)
    B[:, o:, o:] = inp.B_vv
    return np.einsum("Qpq,Qrs->pqrs", B, B)


def _brute_force(inp):
    """Unrestricted (1/3) sum over ALL i,j,k of g, W from dense six-index einsums."""
    o = inp.nocc
    eri = _full_mo(inp)
    ovvv = eri[:o, o:, o:, o:]          # (ia|bd)
    ovoo = eri[:o, o:, :o, :o]          # (ia|jl)
    ovov = eri[:o, o:, :o, o:]          # (ia|jb)
    t1, t2 = inp.t1, inp.t2
    w0 = np.einsum("iabd,kjcd->ijkabc", ovvv, t2) \
        - np.einsum("iajl,lkbc->ijkabc", ovoo, t2)
    W = np.zeros_like(w0)
    for p in itertools.permutations(range(3)):
        # simultaneous permutation of (i,a),(j,b),(k,c)
        axes = list(p) + [3 + x for x in p]
        W += w0.transpose(axes)
    V = W + np.einsum("ia,jbkc->ijkabc", t1, ovov) \
        + np.einsum("jb,iakc->ijkabc", t1, ovov) \
        + np.einsum("kc,iajb->ijkabc", t1, ovov)
    R = 4 * W + W.transpose(0, 1, 2, 4, 5, 3) + W.transpose(0, 1, 2, 5, 3, 4) \
        - 2 * (W.transpose(0, 1, 2, 3, 5, 4) + W.transpose(0, 1, 2, 5, 4, 3)
               + W.transpose(0, 1, 2, 4, 3, 5))
    eo, ev = inp.eps_occ, inp.eps_vir
    D = (eo[:, None, None, None, None, None] + eo[None, :, None, None, None, None]
         + eo[None, None, :, None, None, None] - ev[None, None, None, :, None, None]
         - ev[None, None, None, None, :, None] - ev[None, None, None, None, None, :])
    g = (R * V / D).sum(axis=(3, 4, 5))
    return g.sum() / 3.0, g, W, V


def _abc_driven(inp):
    """The paper's own loop: E = 2 sum_{a>=b>=c} (1/alpha) sum_ijk r3(W)/D V,
    alpha = 6/2/1 (reading G3/G4), r3 = the 4/1/1/-2/-2/-2 pattern applied to ijk."""
    _, _, W, V = _brute_force(inp)
    eo, ev = inp.eps_occ, inp.eps_vir
    E = 0.0
    for a in range(inp.nvir):
        for b in range(a + 1):
            for c in range(b + 1):
                w = W[:, :, :, a, b, c]
                v = V[:, :, :, a, b, c]
                r = 4 * w + w.transpose(1, 2, 0) + w.transpose(2, 0, 1) \
                    - 2 * (w.transpose(0, 2, 1) + w.transpose(2, 1, 0) + w.transpose(1, 0, 2))
                D = (eo[:, None, None] + eo[None, :, None] + eo[None, None, :]
                     - ev[a] - ev[b] - ev[c])
                alpha = 6.0 if a == b == c else (2.0 if (a == b or b == c) else 1.0)
                E += 2.0 * (r * v / D).sum() / alpha
    return E


@pytest.fixture(scope="module")
def small():
    return make_inputs(4, 5, 9, seed=3, t1_std=0.05, t2_std=0.03)


def test_brute_force_six_index(small):
    e_bf, g, W6, V6 = _brute_force(small)
    e, e_trip = orc.t_energy(small, return_triplets=True)
    assert e == pytest.approx(e_bf, rel=1e-12)
    # element-wise W and V for a few triplets, incl. degenerate ones
    for (i, j, k) in [(0, 1, 2), (1, 1, 3), (0, 2, 2), (3, 3, 3), (2, 0, 1)]:
        W = orc.w_triplet(small, i, j, k)
        np.testing.assert_allclose(W, W6[i, j, k], rtol=1e-12, atol=1e-16)
        np.testing.assert_allclose(orc.v_triplet(small, i, j, k, W), V6[i, j, k],
                                   rtol=1e-12, atol=1e-16)
    # per-triplet weights: restricted weighted value == sum of g over distinct orderings / 3
    for n, (i, j, k) in enumerate(orc.triplet_list(small.nocc)):
        perms = set(itertools.permutations((i, j, k)))
        assert e_trip[n] == pytest.approx(sum(g[p] for p in perms) / 3.0,
                                          rel=1e-11, abs=1e-18)


def test_abc_driven_form_of_the_paper(small):
    assert orc.t_energy(small) == pytest.approx(_abc_driven(small), rel=1e-12)


def test_g_symmetric_under_ijk_relabelling(small):
    g012 = orc.g_triplet(small, 0, 1, 2)
    for p in itertools.permutations((0, 1, 2)):
        assert orc.g_triplet(small, *p) == pytest.approx(g012, rel=1e-12)


def test_w_and_v_elements_one_by_one(small):
    rng = np.random.default_rng(0)
    for (i, j, k) in [(0, 1, 3), (2, 2, 3), (1, 3, 3)]:
        W = orc.w_triplet(small, i, j, k)
        V = orc.v_triplet(small, i, j, k, W)
        for _ in range(6):
            a, b, c = (int(x) for x in rng.integers(0, small.nvir, 3))
            assert orc.w_element(small, i, j, k, a, b, c) == pytest.approx(W[a, b, c], rel=1e-11, abs=1e-17)
            assert orc.v_element(small, i, j, k, a, b, c) == pytest.approx(V[a, b, c], rel=1e-11, abs=1e-17)


# ---- P5: each slab against its definition written as explicit loops ---------
def test_slabs_match_explicit_sums_over_Q():
    """(pq|rs) = sum_Q B[Q,p,q] B[Q,r,s] written as plain Python loops on a tiny input (no library contraction:
    a transposed operand or a wrong block in slab_* would fail here)."""
    inp = make_inputs(3, 4, 5, seed=11)
    X, o, v = inp.naux, inp.nocc, inp.nvir
    x, y = 1, 2
    I, O, J = orc.slab_vvov(inp, x), orc.slab_ooov(inp, x, y), orc.slab_ovov(inp, x, y)
    for u in range(v):
        for b in range(v):
            for d in range(v):
                ref = sum(inp.B_ov[Q, x, u] * inp.B_vv[Q, b, d] for Q in range(X))
                assert I[u, b, d] == pytest.approx(ref, rel=1e-13, abs=1e-17)
        for l in range(o):
            ref = sum(inp.B_ov[Q, x, u] * inp.B_oo[Q, y, l] for Q in range(X))
            assert O[l, u] == pytest.approx(ref, rel=1e-13, abs=1e-17)
        for w in range(v):
            ref = sum(inp.B_ov[Q, x, u] * inp.B_ov[Q, y, w] for Q in range(X))
            assert J[u, w] == pytest.approx(ref, rel=1e-13, abs=1e-17)
    # symmetries the definition implies
    np.testing.assert_allclose(I, I.transpose(0, 2, 1), rtol=1e-12, atol=1e-16)
    np.testing.assert_allclose(J, orc.slab_ovov(inp, y, x).T, rtol=1e-13)


# ---- P3: invariants and special cases --------------------------------------
def _scaled(inp, **f):
    out = copy.deepcopy(inp)
    for name, fac in f.items():
        for arr_name in {"t": ["t1", "t2"], "B": ["B_oo", "B_ov", "B_vv"],
                         "eps": ["eps_occ", "eps_vir"], "t1": ["t1"], "t2": ["t2"]}[name]:
            setattr(out, arr_name, getattr(out, arr_name) * fac)
    return out


def test_zero_amplitudes_give_zero(small):
    assert orc.t_energy(_scaled(small, t=0.0)) == 0.0


def test_homogeneity(small):
    e = orc.t_energy(small)
    assert orc.t_energy(_scaled(small, t=1.7)) == pytest.approx(1.7 ** 2 * e, rel=1e-12)
    assert orc.t_energy(_scaled(small, B=1.3)) == pytest.approx(1.3 ** 4 * e, rel=1e-12)
    assert orc.t_energy(_scaled(small, B=-1.0)) == pytest.approx(e, rel=1e-13)
    assert orc.t_energy(_scaled(small, eps=2.5)) == pytest.approx(e / 2.5, rel=1e-12)
    # E[4] quadratic in t2 at t1 = 0
    e4 = orc.t_energy(small, with_t1=False)
    assert orc.t_energy(_scaled(small, t2=3.0), with_t1=False) == pytest.approx(9 * e4, rel=1e-12)
    # E[5] bilinear: linear in t1 at fixed t2
    e5 = e - e4
    e5b = orc.t_energy(_scaled(small, t1=2.0)) - e4
    assert e5b == pytest.approx(2 * e5, rel=1e-10)


def test_orbital_relabelling_invariance(small):
    rng = np.random.default_rng(5)
    po = rng.permutation(small.nocc)
    pv = rng.permutation(small.nvir)
    q = copy.deepcopy(small)
    q.eps_occ = small.eps_occ[po]
    q.eps_vir = small.eps_vir[pv]
    q.t1 = small.t1[np.ix_(po, pv)]
    q.t2 = small.t2[np.ix_(po, po, pv, pv)]
    q.B_oo = small.B_oo[:, po][:, :, po]
    q.B_ov = small.B_ov[:, po][:, :, pv]
    q.B_vv = small.B_vv[:, pv][:, :, pv]
    assert orc.t_energy(q) == pytest.approx(orc.t_energy(small), rel=1e-12)


def test_diagonal_triplets_and_single_pair_vanish(small):
    scale = abs(orc.g_triplet(small, 0, 1, 2))
    for i in range(small.nocc):
        assert abs(orc.g_triplet(small, i, i, i)) < 1e-13 * scale
    one = make_inputs(1, 6, 8, seed=2, t1_std=0.05, t2_std=0.05)
    assert abs(orc.t_energy(one)) < 1e-20


def test_e4_negative_semidefinite(small):
    for (i, j, k) in orc.triplet_list(small.nocc):
        assert orc.g_triplet(small, i, j, k, with_t1=False) <= 1e-18


def test_dropped_term_would_be_caught(small):
    """Sensitivity: a wrong hole sign / missing permutation moves E by >> tolerance."""
    e = orc.t_energy(small)
    q = copy.deepcopy(small)
    q.B_oo = -small.B_oo          # flips only the hole term's sign
    assert abs(orc.t_energy(q) - e) > 1e-3 * abs(e)


# ---- generator (G12) -------------------------------------------------------
def test_generator_recipe_and_symmetries():
    inp = make_config(1)
    assert (inp.nocc, inp.nvir, inp.naux) == (5, 19, 84)
    np.testing.assert_array_equal(inp.t2, inp.t2.transpose(1, 0, 3, 2))
    np.testing.assert_array_equal(inp.B_vv, inp.B_vv.transpose(0, 2, 1))
    np.testing.assert_array_equal(inp.B_oo, inp.B_oo.transpose(0, 2, 1))
    assert np.all(np.diff(inp.eps_occ) >= 0) and np.all(np.diff(inp.eps_vir) >= 0)
    assert -1.5 <= inp.eps_occ.min() and inp.eps_occ.max() <= -0.4
    assert 0.15 <= inp.eps_vir.min() and inp.eps_vir.max() <= 3.0
    # same stream reproduced by hand
    rng = np.random.default_rng(1001)
    G = rng.normal(0.0, 0.1, size=(84, 24, 24))
    Bs = 0.5 * (G + G.transpose(0, 2, 1))
    np.testing.assert_allclose(inp.B_ov, Bs[:, :5, 5:], rtol=0, atol=1e-17)
    eo = np.sort(rng.uniform(-1.5, -0.4, 5))
    np.testing.assert_array_equal(inp.eps_occ, eo)
    for a in inp.arrays():
        assert a.flags.c_contiguous and a.dtype == np.float64


def test_config1_magnitude():
    # SURVEY.md §8(c) "Magnitudes": config 1 E(T) is O(-1) Eh on this generator
    e = orc.t_energy(make_config(1))
    assert -5.0 < e < -0.1


def test_sample_triplets_cover_classes():
    s = sample_triplets(40, 16, seed=9)
    assert len(s) == 16 and len(set(s)) == 16
    assert all(i <= j <= k for i, j, k in s)
    assert any(i == j < k for i, j, k in s) and any(i < j == k for i, j, k in s)
    assert any(i < j < k for i, j, k in s) and any(i == j == k for i, j, k in s)


# ---- NEXT-3: occupied-virtual Fock block (Eqs. (5),(7)) ----
def test_fock_term_is_linear_in_f_and_vanishes_at_zero():
    inp = make_inputs(3, 5, 7, seed=21, t1_std=0.05, t2_std=0.05, f_std=0.1)
    canon = copy.copy(inp); canon.f_ov = None
    zero = copy.copy(inp); zero.f_ov = np.zeros_like(inp.f_ov)
    twice = copy.copy(inp); twice.f_ov = 2.0 * inp.f_ov
    e0, e1, e2 = orc.t_energy(canon), orc.t_energy(inp), orc.t_energy(twice)
    assert orc.t_energy(zero) == e0
    assert abs(e1 - e0) > 1e-6 * abs(e0)
    assert (e2 - e0) == pytest.approx(2.0 * (e1 - e0), rel=1e-10)
    # E_F is bilinear in (f, t2) x (W ~ t2): scaling t2 by s scales it by s^2, t1 does not enter it
    not1 = copy.copy(inp); not1.t1 = np.zeros_like(inp.t1)
    not1c = copy.copy(canon); not1c.t1 = np.zeros_like(inp.t1)
    assert (orc.t_energy(not1) - orc.t_energy(not1c)) == pytest.approx(e1 - e0, rel=1e-10)


def test_fock_term_brute_force_and_elements():
    """E_F against a dense six-index contraction sum_{ijkabc} R[W] f[k,c] t2[i,j,a,b] / D (x3 by symmetry / 3)."""
    inp = make_inputs(3, 4, 6, seed=22, t1_std=0.05, t2_std=0.05, f_std=0.1)
    canon = copy.copy(inp); canon.f_ov = None
    o, v = inp.nocc, inp.nvir
    W6 = np.zeros((o, o, o, v, v, v))
    for i, j, k in itertools.product(range(o), repeat=3):
        W6[i, j, k] = orc.w_triplet(inp, i, j, k)
    R6 = (4 * W6 + W6.transpose(0, 1, 2, 4, 5, 3) + W6.transpose(0, 1, 2, 5, 3, 4)
          - 2 * (W6.transpose(0, 1, 2, 3, 5, 4) + W6.transpose(0, 1, 2, 5, 4, 3) + W6.transpose(0, 1, 2, 4, 3, 5)))
    eo, ev = inp.eps_occ, inp.eps_vir
    D6 = (eo[:, None, None, None, None, None] + eo[None, :, None, None, None, None]
          + eo[None, None, :, None, None, None] - ev[None, None, None, :, None, None]
          - ev[None, None, None, None, :, None] - ev[None, None, None, None, None, :])
    # the three f*t2 terms are images of one another under simultaneous (occ, vir) relabelling, and R/D is
    # invariant under it: (1/3) sum_all 3 * [R/D * f[k,c] t2[i,j,a,b]]
    ef = np.einsum("ijkabc,kc,ijab->", R6 / D6, inp.f_ov, inp.t2)
    assert (orc.t_energy(inp) - orc.t_energy(canon)) == pytest.approx(ef, rel=1e-10)
    W = orc.w_triplet(inp, 0, 1, 2)
    V = orc.v_triplet(inp, 0, 1, 2, W)
    for (a, b, c) in [(0, 1, 2), (3, 3, 1), (2, 0, 0)]:
        assert orc.v_element(inp, 0, 1, 2, a, b, c) == pytest.approx(V[a, b, c], rel=1e-11, abs=1e-16)
