"""CPU ORACLE for the closed-shell DF-MP2 correlation energy.  TEST INFRASTRUCTURE.

Not part of the product: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import it.  It
shares no code with ``paper_2502_17963_b200/`` (only the seeded input generator
``bqc_inputs`` serves both, and that module holds none of the method's
arithmetic).

What it follows
---------------
PAPER.md:252-258 (§2.3, Eq. (1)), SURVEY.md §8(f) NEXT-4:

    E_MP2 = sum_{i,j,a,b} (ia|jb) [ 2 (ia|jb) - (ib|ja) ] / (e_i + e_j - e_a - e_b)     Eq. (1)

with i, j over the doubly occupied and a, b over the virtual orbitals, the sum
unrestricted over all four indices (reading M1: the paper prints a bare "sum";
the unrestricted closed-shell sum is the textbook one and is what the
first-principles pin fixes), and density-fitted integrals
(ia|jb) = sum_Q B_ov[Q,i,a] B_ov[Q,j,b] ("computed in advance in DF
form"; exact DF as in BASELINE.json configs[0]).  The denominator is evaluated
on the fly from the orbital energies, never stored as a rank-4 tensor
(PAPER.md:256).

    J_ij[a,b] = (ia|jb)                               one v x v matrix per occupied pair
    e_ij      = sum_{a,b} J_ij[a,b] (2 J_ij[a,b] - J_ij[b,a]) / (e_i + e_j - e_a - e_b)
    E_MP2     = sum_{i,j} e_ij            (e_ij = e_ji, so also sum_{i<=j} (2 - d_ij) e_ij)

Arithmetic is FP64 NumPy; ``@`` is the library contraction primitive of the one
contraction step.  No blocking or reordering beyond the lines above.  Pinned by
``tests/test_mp2_oracle_pins.py`` (``-m "not gpu"``): a second-quantised
second-order perturbation energy that uses no index formula, a hand-computed
closed form, the opposite-spin / same-spin decomposition, scaling laws,
relabelling invariance and brute-force loops.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def ovov_pair(inp, i, j):
    """J_ij[a,b] = (ia|jb) = sum_Q B_ov[Q,i,a] B_ov[Q,j,b]."""
    return inp.B_ov[:, i, :].T @ inp.B_ov[:, j, :]


def pair_energy(inp, i, j):
    """e_ij of Eq. (1): the (i,j) slice of the unrestricted sum."""
    J = ovov_pair(inp, i, j)
    D = inp.eps_occ[i] + inp.eps_occ[j] - inp.eps_vir[:, None] - inp.eps_vir[None, :]
    return float(np.sum(J * (2.0 * J - J.T) / D, dtype=np.longdouble))


def pair_energies(inp):
    """[nocc, nocc] matrix of e_ij."""
    o = inp.nocc
    e = np.zeros((o, o))
    for i in range(o):
        for j in range(o):
            e[i, j] = pair_energy(inp, i, j)
    return e


def mp2_energy(inp):
    """E_MP2 of Eq. (1): sum over all ordered occupied pairs, in index order."""
    return float(np.sum(pair_energies(inp), dtype=np.longdouble))
