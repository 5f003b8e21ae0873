"""Seeded input generators (no (T) arithmetic lives here).

Recipe (BASELINE.json `configs`, reading G12 of SURVEY.md §8(c)):

* one NumPy ``default_rng(seed)`` (PCG64) stream, draws in this order, each a
  full-array draw in C order:
    1. ``G_B``   [naux, n, n]  N(0, 0.1)   over all n = nocc + nvir MOs,
       ``B = (G_B + G_B^T(p<->q)) / 2``; ``B_oo, B_ov, B_vv`` are contiguous
       copies of its blocks (occupied MOs first);
    2. ``eps_occ`` [nocc] uniform[-1.5, -0.4], sorted ascending;
    3. ``eps_vir`` [nvir] uniform[0.15, 3.0], sorted ascending;
    4. ``t1``    [nocc, nvir] N(0, t1_std);
    5. ``G_t2``  [nocc, nocc, nvir, nvir] N(0, t2_std),
       ``t2 = (G_t2 + G_t2.transpose(1, 0, 3, 2)) / 2``;
    6. only when ``f_std > 0`` (non-canonical reference):
       ``f_ov`` [nocc, nvir] N(0, f_std), drawn last so draws 1-5 do not change.
* integrals are *defined* as (pq|rs) = sum_Q B[Q,p,q] B[Q,r,s]  (exact DF).
* "sliced" recipe (config 9, the paper's largest CCSD(T) size, 117 GB of inputs): the same distributions and
  symmetrisations, but every Q-slice of B and every t2[i] slab has its own PCG64 stream,
  ``default_rng([seed, 1, q])`` / ``default_rng([seed, 3, i])`` (eps_occ, eps_vir, t1 from
  ``default_rng([seed, 2])`` in that order), so that the slices can be drawn in parallel and B is never held
  as one [naux, n, n] array.

These are synthetic stand-ins shaped like the paper's water-cluster cc-pVDZ
workloads (24 orbitals, 5 occupied per water).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class TInputs:
    """Inputs of one (T) evaluation.  All arrays FP64, C-contiguous."""
    nocc: int
    nvir: int
    naux: int
    eps_occ: np.ndarray   # [nocc]
    eps_vir: np.ndarray   # [nvir]
    t1: np.ndarray        # [nocc, nvir]
    t2: np.ndarray        # [nocc, nocc, nvir, nvir], t2[i,j,a,b] == t2[j,i,b,a]
    B_oo: np.ndarray      # [naux, nocc, nocc]
    B_ov: np.ndarray      # [naux, nocc, nvir]
    B_vv: np.ndarray      # [naux, nvir, nvir]
    name: str = ""
    f_ov: np.ndarray | None = None   # [nocc, nvir] occupied-virtual Fock block; None = canonical RHF

    def arrays(self):
        return (self.eps_occ, self.eps_vir, self.t1, self.t2,
                self.B_oo, self.B_ov, self.B_vv)

    def nbytes(self) -> int:
        return sum(a.nbytes for a in self.arrays())


# BASELINE.json configs[0..4]: (nocc, nvir, naux, t2_std, seed)
CONFIGS = {
    1: dict(nocc=5, nvir=19, naux=84, t2_std=1e-2, seed=1001),
    2: dict(nocc=20, nvir=76, naux=336, t2_std=1e-2, seed=1002),
    3: dict(nocc=40, nvir=152, naux=672, t2_std=1e-2, seed=1003),
    4: dict(nocc=80, nvir=304, naux=1344, t2_std=5e-3, seed=1004),
    5: dict(nocc=100, nvir=380, naux=1680, t2_std=5e-3, seed=1005),
    # larger-basis shapes (same generator).  The paper's water clusters in
    # cc-pVTZ / cc-pVQZ have 58 / 115 orbitals and 5 occupied per water (8.6 % / 4.3 %
    # occupied); naux = 3.5 x orbitals as in configs 1-5.
    6: dict(nocc=20, nvir=212, naux=812, t2_std=1e-2, seed=1006),    # 4 waters, cc-pVTZ-shaped
    7: dict(nocc=10, nvir=220, naux=805, t2_std=1e-2, seed=1007),    # 2 waters, cc-pVQZ-shaped
    8: dict(nocc=40, nvir=424, naux=1624, t2_std=5e-3, seed=1008),   # 8 waters, cc-pVTZ-shaped
    # PAPER.md:381 "capable of handling up to 1 380 orbitals": 12 waters, cc-pVQZ-shaped (115 orbitals and
    # 5 occupied per water), naux = 3.5 x orbitals.  117 GB of inputs: the sliced recipe above.
    9: dict(nocc=60, nvir=1320, naux=4830, t2_std=5e-3, seed=1009, recipe="sliced"),
}


def make_inputs(nocc: int, nvir: int, naux: int, seed: int,
                t1_std: float = 1e-3, t2_std: float = 1e-2,
                b_std: float = 0.1, name: str = "", f_std: float = 0.0) -> TInputs:
    """Generate one seeded input set following the G12 recipe above."""
    rng = np.random.default_rng(seed)
    n = nocc + nvir
    B = rng.normal(0.0, b_std, size=(naux, n, n))
    # in-place symmetrisation in p<->q, one Q-slice at a time (config 5 is 3 GB)
    for q in range(naux):
        s = B[q]
        s += s.T.copy()
        s *= 0.5
    B_oo = np.ascontiguousarray(B[:, :nocc, :nocc])
    B_ov = np.ascontiguousarray(B[:, :nocc, nocc:])
    B_vv = np.ascontiguousarray(B[:, nocc:, nocc:])
    del B
    eps_occ = np.sort(rng.uniform(-1.5, -0.4, size=nocc))
    eps_vir = np.sort(rng.uniform(0.15, 3.0, size=nvir))
    t1 = rng.normal(0.0, t1_std, size=(nocc, nvir))
    t2 = rng.normal(0.0, t2_std, size=(nocc, nocc, nvir, nvir))
    # t2 <- (G + G.transpose(1,0,3,2)) / 2 without a second full-size copy
    for i in range(nocc):
        for j in range(i, nocc):
            if i == j:
                blk = t2[i, i]
                blk += blk.T.copy()
                blk *= 0.5
            else:
                a = t2[i, j]
                b = t2[j, i]
                a += b.T
                a *= 0.5
                b[...] = a.T
    f_ov = rng.normal(0.0, f_std, size=(nocc, nvir)) if f_std > 0.0 else None
    return TInputs(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv,
                   name=name or f"o{nocc}v{nvir}x{naux}s{seed}", f_ov=f_ov)


def _symmetrise_t2(t2: np.ndarray) -> None:
    """t2 <- (G + G.transpose(1,0,3,2)) / 2 in place, without a second full-size copy."""
    nocc = t2.shape[0]
    for i in range(nocc):
        for j in range(i, nocc):
            if i == j:
                blk = t2[i, i]
                blk += blk.T.copy()
                blk *= 0.5
            else:
                a = t2[i, j]
                b = t2[j, i]
                a += b.T
                a *= 0.5
                b[...] = a.T


def make_inputs_sliced(nocc: int, nvir: int, naux: int, seed: int, t1_std: float = 1e-3,
                       t2_std: float = 1e-2, b_std: float = 0.1, name: str = "", threads: int = 0) -> TInputs:
    """The "sliced" recipe of the module docstring: one stream per Q-slice of B and per t2[i] slab, drawn by
    a thread pool (NumPy releases the GIL while it fills), block arrays written in place."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    n = nocc + nvir
    B_oo = np.empty((naux, nocc, nocc))
    B_ov = np.empty((naux, nocc, nvir))
    B_vv = np.empty((naux, nvir, nvir))

    def b_slice(q):
        g = np.random.default_rng([seed, 1, q]).normal(0.0, b_std, size=(n, n))
        g += g.T.copy()
        g *= 0.5
        B_oo[q] = g[:nocc, :nocc]
        B_ov[q] = g[:nocc, nocc:]
        B_vv[q] = g[nocc:, nocc:]

    t2 = np.empty((nocc, nocc, nvir, nvir))

    def t2_slab(i):
        t2[i] = np.random.default_rng([seed, 3, i]).normal(0.0, t2_std, size=(nocc, nvir, nvir))

    with ThreadPoolExecutor(max_workers=threads or (os.cpu_count() or 1)) as ex:
        list(ex.map(b_slice, range(naux)))
        list(ex.map(t2_slab, range(nocc)))
    rng = np.random.default_rng([seed, 2])
    eps_occ = np.sort(rng.uniform(-1.5, -0.4, size=nocc))
    eps_vir = np.sort(rng.uniform(0.15, 3.0, size=nvir))
    t1 = rng.normal(0.0, t1_std, size=(nocc, nvir))
    _symmetrise_t2(t2)
    return TInputs(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv,
                   name=name or f"o{nocc}v{nvir}x{naux}s{seed}sliced")


def make_config(idx: int, **overrides) -> TInputs:
    """BASELINE.json configs[idx-1] (idx = 1..5); idx = 6..8: the larger-basis shapes of NEXT-2; 9: the paper's
    largest CCSD(T) size (sliced recipe)."""
    c = dict(CONFIGS[idx])
    c.update(overrides)
    if c.get("recipe") == "sliced":
        return make_inputs_sliced(c["nocc"], c["nvir"], c["naux"], c["seed"], t1_std=c.get("t1_std", 1e-3),
                                  t2_std=c["t2_std"], name=f"config{idx}")
    return make_inputs(c["nocc"], c["nvir"], c["naux"], c["seed"],
                       t1_std=c.get("t1_std", 1e-3), t2_std=c["t2_std"],
                       name=f"config{idx}", f_std=c.get("f_std", 0.0))


def worked_example(nocc: int, nvir: int, naux: int) -> TInputs:
    """Deterministic closed-form inputs of SURVEY.md §8(c) P2 (no RNG)."""
    n = nocc + nvir
    Q = np.arange(naux, dtype=np.float64)[:, None, None]
    p = np.arange(n, dtype=np.float64)[None, :, None]
    q = np.arange(n, dtype=np.float64)[None, None, :]
    B = 0.1 * np.cos(1.0 + 0.7 * Q + 1.3 * (p + q) + 0.37 * p * q)
    i = np.arange(nocc, dtype=np.float64)
    a = np.arange(nvir, dtype=np.float64)
    eps_occ = -1.5 + 1.1 * (i + 0.5) / nocc
    eps_vir = 0.15 + 2.85 * (a + 0.5) / nvir
    t1 = 0.05 * np.sin(1.0 + 2.0 * i[:, None] + 3.0 * a[None, :])
    I = i[:, None, None, None]
    J = i[None, :, None, None]
    A = a[None, None, :, None]
    Bv = a[None, None, None, :]
    t2 = 0.01 * np.cos(0.3 + 1.1 * (I + J) + 0.7 * (A + Bv)
                       + 0.5 * (I * A + J * Bv) + 0.9 * (I * Bv + J * A))
    return TInputs(nocc, nvir, naux, eps_occ, eps_vir,
                   np.ascontiguousarray(t1), np.ascontiguousarray(t2),
                   np.ascontiguousarray(B[:, :nocc, :nocc]),
                   np.ascontiguousarray(B[:, :nocc, nocc:]),
                   np.ascontiguousarray(B[:, nocc:, nocc:]),
                   name=f"worked_o{nocc}v{nvir}x{naux}")


def sample_triplets(nocc: int, count: int, seed: int):
    """Seeded random subset of occupied triplets i<=j<=k.

    Always contains one i=j<k, one i<j=k, one i<j<k and one diagonal triplet
    (when nocc allows); the rest are uniform draws without repetition.
    """
    rng = np.random.default_rng(seed)
    out = []
    if nocc >= 2:
        out += [(0, 0, nocc - 1), (0, nocc - 1, nocc - 1)]
    if nocc >= 3:
        out += [(0, nocc // 2, nocc - 1)]
    out += [(nocc // 2, nocc // 2, nocc // 2)]
    seen = set(out)
    guard = 0
    while len(out) < count and guard < 100000:
        guard += 1
        t = tuple(sorted(int(x) for x in rng.integers(0, nocc, size=3)))
        if t not in seen:
            seen.add(t)
            out.append(t)
    return out[:max(count, 1)]
