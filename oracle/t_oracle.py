"""CPU ORACLE for the closed-shell RHF (T) energy correction.  TEST INFRASTRUCTURE.

This file is the plain, slow, obviously-correct statement of what the CUDA path
must compute.  It is NOT part of the product: only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import it.  It shares no code with
``paper_2502_17963_b200/`` (only the seeded input generator ``bqc_inputs`` serves
both, and that module holds none of the method's arithmetic).

What it follows
---------------
PAPER.md:288-305 (§2.4.2, Eqs. (2)-(7)) with the readings G1-G7 of SURVEY.md
§8(c) / DESIGN.md "Readings of the paper":

  W_ijk[a,b,c] = sum over the 6 simultaneous permutations
                 ((x1,u1),(x2,u2),(x3,u3)) of ((i,a),(j,b),(k,c)) of
                   + sum_d (x1 u1 | u2 d) * t2[x3, x2, u3, d]         Eq. (2), particle
                   - sum_l (x1 u1 | x2 l) * t2[l,  x3, u2, u3]        Eq. (2), hole (G1)
  V_ijk[a,b,c] = W_ijk[a,b,c] + t1[i,a](jb|kc) + t1[j,b](ia|kc) + t1[k,c](ia|jb)
                                                          Eqs. (6),(7) (G6)
  R_ijk[a,b,c] = 4 W[a,b,c] + W[b,c,a] + W[c,a,b]
                 - 2 (W[a,c,b] + W[c,b,a] + W[b,a,c])             Eq. (3) numerator (G2)
  D_ijk[a,b,c] = e_i + e_j + e_k - e_a - e_b - e_c                  Eq. (3) denominator
  g(i,j,k)     = sum_{a,b,c} R V / D                                Eq. (4)
  E(T)         = sum_{i<=j<=k} (2 - d_ij - d_jk) g(i,j,k)           (G3, G4)

Integrals are exact density fitting, (pq|rs) = sum_Q B[Q,p,q] B[Q,r,s]
(BASELINE.json configs[0]).  The Fock term of Eqs. (5),(7)
vanishes for canonical RHF (G7); when the input carries an occupied-virtual
Fock block ``f_ov`` V gains
f[i,a] t2[j,k,b,c] + f[j,b] t2[i,k,a,c] + f[k,c] t2[i,j,a,b]  (reading G15).

The paper's own loop order ("abc-driven") is
written out as well — ``w_virtual_triple`` / ``v_virtual_triple`` /
``e_virtual_triple`` / ``t_energy_abc``: one virtual triple a<=b<=c at a time, all
o^3 occupied triples inside, E = 2 sum_{a<=b<=c} (1/alpha) sum_ijk [r3_ijk(W)/D] V
with alpha = 1/2/6 (reading G3).  Pinned by ``tests/test_abc_oracle_pins.py``.

Arithmetic is FP64 NumPy.  ``numpy.einsum`` / ``@`` serve as the library
contraction primitive of each step; there is no blocking, fusion or reordering
beyond the equations above.  Every function is pinned by ``tests/`` (``-m "not
gpu"``): a first-principles second-quantised evaluation (P1), the worked
examples of SURVEY.md §8(c) P2 (``tests/golden/``), brute-force six-index
einsum, invariants and special cases.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import itertools

import numpy as np

_PERMS = list(itertools.permutations((0, 1, 2)))


# --------------------------------------------------------------------------
# DF integrals (SURVEY.md §8 slab definitions)
# --------------------------------------------------------------------------
def slab_vvov(inp, x):
    """I_x[u,b,d] = (x u | b d) = sum_Q B_ov[Q,x,u] B_vv[Q,b,d]."""
    return np.einsum("Qu,Qbd->ubd", inp.B_ov[:, x, :], inp.B_vv, optimize=True)


def slab_ooov(inp, x, y):
    """O_xy[l,u] = (x u | y l) = sum_Q B_ov[Q,x,u] B_oo[Q,y,l]."""
    return np.einsum("Qu,Ql->lu", inp.B_ov[:, x, :], inp.B_oo[:, y, :])


def slab_ovov(inp, x, y):
    """J_xy[u,w] = (x u | y w) = sum_Q B_ov[Q,x,u] B_ov[Q,y,w]."""
    return np.einsum("Qu,Qw->uw", inp.B_ov[:, x, :], inp.B_ov[:, y, :])


# --------------------------------------------------------------------------
# Eq. (2): W intermediate of one occupied triplet
# --------------------------------------------------------------------------
def w_triplet(inp, i, j, k, slabs=None):
    """W_ijk[a,b,c] of Eq. (2) (reading G1/G5).

    `slabs` may carry precomputed {x: I_x}; it is a cache only.
    """
    occ = (i, j, k)
    v = inp.nvir
    W = np.zeros((v, v, v))
    for perm in _PERMS:
        x1, x2, x3 = occ[perm[0]], occ[perm[1]], occ[perm[2]]
        I1 = slabs[x1] if slabs is not None else slab_vvov(inp, x1)
        # particle: sum_d (x1 u1|u2 d) t2[x3,x2,u3,d]
        w0 = np.einsum("pqd,rd->pqr", I1, inp.t2[x3, x2], optimize=True)
        # hole:   - sum_l (x1 u1|x2 l) t2[l,x3,u2,u3]
        w0 -= np.einsum("lp,lqr->pqr", slab_ooov(inp, x1, x2), inp.t2[:, x3],
                        optimize=True)
        # w0 is indexed [u1,u2,u3]; u_m is the virtual paired with occ[perm[m]],
        # i.e. axis m of w0 is axis perm[m] of W[a,b,c].
        W += np.transpose(w0, np.argsort(perm))
    return W


def v_triplet(inp, i, j, k, W):
    """V = W + t1 (ov|ov) terms (Eqs. (6),(7), reading G6).

    Non-canonical reference (inp.f_ov given; Eqs. (5),(7), reading G15): the x-term
    x_k F_ck = 0.5 P sum_ij t_ij^ab v_ijk F_ck adds, by the same argument as G6,
    f[i,a] t2[j,k,b,c] + f[j,b] t2[i,k,a,c] + f[k,c] t2[i,j,a,b] to V.
    """
    t1 = inp.t1
    V = W.copy()
    V += t1[i][:, None, None] * slab_ovov(inp, j, k)[None, :, :]
    V += t1[j][None, :, None] * slab_ovov(inp, i, k)[:, None, :]
    V += t1[k][None, None, :] * slab_ovov(inp, i, j)[:, :, None]
    f = getattr(inp, "f_ov", None)
    if f is not None:
        V += f[i][:, None, None] * inp.t2[j, k][None, :, :]
        V += f[j][None, :, None] * inp.t2[i, k][:, None, :]
        V += f[k][None, None, :] * inp.t2[i, j][:, :, None]
    return V


def r_of_w(W):
    """Eq. (3) numerator, six terms (reading G2).

    X.transpose(2,0,1)[a,b,c] = X[b,c,a];  X.transpose(1,2,0)[a,b,c] = X[c,a,b].
    """
    return (4.0 * W + W.transpose(2, 0, 1) + W.transpose(1, 2, 0)
            - 2.0 * (W.transpose(0, 2, 1) + W.transpose(2, 1, 0)
                     + W.transpose(1, 0, 2)))


def d_triplet(inp, i, j, k):
    """Eq. (3) denominator D_ijk[a,b,c]."""
    e = inp.eps_vir
    dijk = inp.eps_occ[i] + inp.eps_occ[j] + inp.eps_occ[k]
    return dijk - e[:, None, None] - e[None, :, None] - e[None, None, :]


def triplet_weight(i, j, k):
    """(2 - delta_ij - delta_jk) for i<=j<=k (reading G3)."""
    return 2.0 - (1.0 if i == j else 0.0) - (1.0 if j == k else 0.0)


def g_triplet(inp, i, j, k, slabs=None, with_t1=True):
    """g(i,j,k) = sum_abc R V / D (Eq. (4)); unweighted."""
    W = w_triplet(inp, i, j, k, slabs)
    V = v_triplet(inp, i, j, k, W) if with_t1 else W
    x = r_of_w(W) * V / d_triplet(inp, i, j, k)
    return float(np.sum(x.astype(np.longdouble)))


def e_triplet(inp, i, j, k, slabs=None, with_t1=True):
    """Weighted per-triplet contribution e_ijk = (2-d_ij-d_jk) g(i,j,k), i<=j<=k."""
    assert i <= j <= k
    return triplet_weight(i, j, k) * g_triplet(inp, i, j, k, slabs, with_t1)


def num_triplets(nocc):
    return nocc * (nocc + 1) * (nocc + 2) // 6


def triplet_list(nocc):
    """All i<=j<=k in lexicographic order (the library's triplet index order)."""
    return [(i, j, k) for i in range(nocc) for j in range(i, nocc)
            for k in range(j, nocc)]


def t_energy(inp, with_t1=True, return_triplets=False, cache_slabs=True):
    """E(T) = sum_{i<=j<=k} e_ijk, summed in triplet-index order."""
    slabs = None
    if cache_slabs:
        slabs = {x: slab_vvov(inp, x) for x in range(inp.nocc)}
    e = np.zeros(num_triplets(inp.nocc))
    for n, (i, j, k) in enumerate(triplet_list(inp.nocc)):
        e[n] = e_triplet(inp, i, j, k, slabs, with_t1)
    total = float(np.sum(e.astype(np.longdouble)))
    return (total, e) if return_triplets else total


# --------------------------------------------------------------------------
# The paper's abc-driven loop (SURVEY.md §8(c) "Passages followed",
# §8(f) NEXT-2): one virtual triple a,b,c at a time, o^3 tensors inside
#     E = 2 sum_{a<=b<=c} (1/alpha) sum_ijk [r3_ijk(W) / D] V,
# alpha = 1 / 2 / 6 for three distinct / exactly two equal / three equal virtuals
# (reading G3), r3 the 4/1/1/-2/-2/-2 pattern of Eq. (3) applied to ijk.
# --------------------------------------------------------------------------
def w_virtual_triple(inp, a, b, c):
    """W^{abc}[i,j,k] of Eq. (2) for one virtual triple and all occupied i,j,k."""
    vir = (a, b, c)
    o = inp.nocc
    W = np.zeros((o, o, o))
    for perm in _PERMS:
        u1, u2, u3 = vir[perm[0]], vir[perm[1]], vir[perm[2]]
        # particle: sum_d (x1 u1|u2 d) t2[x3,x2,u3,d]
        ovvv = np.einsum("Qx,Qd->xd", inp.B_ov[:, :, u1], inp.B_vv[:, u2, :])
        w0 = np.einsum("xd,zyd->xyz", ovvv, inp.t2[:, :, u3, :], optimize=True)
        # hole:   - sum_l (x1 u1|x2 l) t2[l,x3,u2,u3]
        ovoo = np.einsum("Qx,Qyl->xyl", inp.B_ov[:, :, u1], inp.B_oo, optimize=True)
        w0 -= np.einsum("xyl,lz->xyz", ovoo, inp.t2[:, :, u2, u3], optimize=True)
        # w0 is indexed [x1,x2,x3]; x_m is the occupied paired with vir[perm[m]],
        # i.e. axis m of w0 is axis perm[m] of W[i,j,k].
        W += np.transpose(w0, np.argsort(perm))
    return W


def v_virtual_triple(inp, a, b, c, W):
    """V^{abc}[i,j,k] = W + t1 (ov|ov) terms (+ the Fock term), Eqs. (5)-(7)."""
    t1 = inp.t1
    J = lambda u, w: np.einsum("Qx,Qy->xy", inp.B_ov[:, :, u], inp.B_ov[:, :, w])  # (x u|y w)
    V = W.copy()
    V += t1[:, a][:, None, None] * J(b, c)[None, :, :]
    V += t1[:, b][None, :, None] * J(a, c)[:, None, :]
    V += t1[:, c][None, None, :] * J(a, b)[:, :, None]
    f = getattr(inp, "f_ov", None)
    if f is not None:
        V += f[:, a][:, None, None] * inp.t2[:, :, b, c][None, :, :]
        V += f[:, b][None, :, None] * inp.t2[:, :, a, c][:, None, :]
        V += f[:, c][None, None, :] * inp.t2[:, :, a, b][:, :, None]
    return V


def e_virtual_triple(inp, a, b, c, with_t1=True):
    """(2/alpha) sum_ijk r3_ijk(W) V / D for a<=b<=c: the abc-driven contribution."""
    assert a <= b <= c
    W = w_virtual_triple(inp, a, b, c)
    V = v_virtual_triple(inp, a, b, c, W) if with_t1 else W
    e = inp.eps_occ
    D = (e[:, None, None] + e[None, :, None] + e[None, None, :]
         - inp.eps_vir[a] - inp.eps_vir[b] - inp.eps_vir[c])
    alpha = 6.0 if a == b == c else (2.0 if (a == b or b == c) else 1.0)
    x = r_of_w(W) * V / D
    return (2.0 / alpha) * float(np.sum(x.astype(np.longdouble)))


def t_energy_abc(inp, with_t1=True, return_triples=False):
    """E(T) by the abc-driven loop, summed in virtual-triple index order."""
    trip = triplet_list(inp.nvir)
    e = np.zeros(len(trip))
    for n, (a, b, c) in enumerate(trip):
        e[n] = e_virtual_triple(inp, a, b, c, with_t1)
    total = float(np.sum(e.astype(np.longdouble)))
    return (total, e) if return_triples else total


# --------------------------------------------------------------------------
# One-by-one sampled outputs for sizes where a whole triplet is too slow
# --------------------------------------------------------------------------
def _eri_ovvv(inp, x, u, b):
    """(x u | b :)  -> [nvir] vector over d."""
    return np.einsum("Q,Qd->d", inp.B_ov[:, x, u], inp.B_vv[:, b, :])


def _eri_ovoo(inp, x, u, y):
    """(x u | y :)  -> [nocc] vector over l."""
    return np.einsum("Q,Ql->l", inp.B_ov[:, x, u], inp.B_oo[:, y, :])


def w_element(inp, i, j, k, a, b, c):
    """One element W_ijk[a,b,c] straight from Eq. (2): 6 + 6 dot products."""
    occ = (i, j, k)
    vir = (a, b, c)
    w = 0.0
    for perm in _PERMS:
        (x1, u1), (x2, u2), (x3, u3) = [(occ[m], vir[m]) for m in perm]
        w += float(_eri_ovvv(inp, x1, u1, u2) @ inp.t2[x3, x2, u3, :])
        w -= float(_eri_ovoo(inp, x1, u1, x2) @ inp.t2[:, x3, u2, u3])
    return w


def v_element(inp, i, j, k, a, b, c, w=None):
    """One element V_ijk[a,b,c]."""
    if w is None:
        w = w_element(inp, i, j, k, a, b, c)
    B = inp.B_ov
    jbkc = float(B[:, j, b] @ B[:, k, c])
    iakc = float(B[:, i, a] @ B[:, k, c])
    iajb = float(B[:, i, a] @ B[:, j, b])
    val = w + inp.t1[i, a] * jbkc + inp.t1[j, b] * iakc + inp.t1[k, c] * iajb
    f = getattr(inp, "f_ov", None)
    if f is not None:
        val += (f[i, a] * inp.t2[j, k, b, c] + f[j, b] * inp.t2[i, k, a, c]
                + f[k, c] * inp.t2[i, j, a, b])
    return val
