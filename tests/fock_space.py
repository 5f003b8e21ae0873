"""First-principles (second-quantised) evaluation of the closed-shell (T) energy.

Pin P1 of SURVEY.md §8(c): uses NO index formula of PAPER.md Eqs. (2)-(7).
Jordan-Wigner matrices on the full Fock space of 2(o+v) spin orbitals;

    E_pq  = sum_sigma a+_{p sigma} a_{q sigma}
    H2    = 1/2 sum_pqrs (pq|rs) (E_pq E_rs - delta_qr E_ps)
    u_pq  = sum_i [2 (pq|ii) - (pi|iq)]            (HF mean field of the occupied space)
    W_N   = H2 - sum_pq u_pq E_pq                   (fluctuation potential)
    T1    = sum_ia t1[i,a] E_ai ;  T2 = 1/2 sum_ijab t2[i,j,a,b] E_ai E_bj
    R3    = diag(1/D) on triply excited determinants, D = sum eps_holes - sum eps_particles
    E[4]  = <0| T2+ W_N R3 W_N T2 |0>,   E[5] = <0| T1+ W_N R3 W_N T2 |0>,
    E(T)  = E[4] + E[5]
Non-canonical reference (Eqs. (5),(7)): with an occupied-virtual
Fock block f_ov the fluctuation potential gains the one-body operator F_ov = sum_ia f[i,a] (E_ia + E_ai) and
    E[F]  = <0| T2+ F_ov R3 W_N T2 |0>,   E(T) = E[4] + E[5] + E[F].
(textbook CCSD(T): Raghavachari et al. 1989; the closed-shell index formula the
paper optimises, PAPER.md:288 ref. 62, must reproduce these numbers.)
"""
import numpy as np
import scipy.sparse as sp


def _jw_annihilators(nso):
    a1 = sp.csr_matrix(np.array([[0.0, 1.0], [0.0, 0.0]]))
    z = sp.csr_matrix(np.diag([1.0, -1.0]))
    eye = sp.identity(2, format="csr")
    ops = []
    for s in range(nso):
        m = sp.identity(1, format="csr")
        for t in range(nso):
            m = sp.kron(m, z if t < s else (a1 if t == s else eye), format="csr")
        ops.append(m)
    return ops


def _model(inp):
    """(E_pq, apply_WN, |HF>, eps, nso) of the model Hamiltonian H0 = sum_p eps_p E_pp, H = H0 + W_N."""
    o, v = inp.nocc, inp.nvir
    n = o + v
    nso = 2 * n
    dim = 1 << nso
    a = _jw_annihilators(nso)
    ad = [m.T.tocsr() for m in a]
    E = [[sum(ad[2 * p + s] @ a[2 * q + s] for s in range(2)).tocsr()
          for q in range(n)] for p in range(n)]

    # full MO DF factor and Mulliken integrals (pq|rs) = sum_Q B[Q,p,q] B[Q,r,s]
    B = np.zeros((inp.naux, n, n))
    B[:, :o, :o] = inp.B_oo
    B[:, :o, o:] = inp.B_ov
    B[:, o:, :o] = inp.B_ov.transpose(0, 2, 1)
    B[:, o:, o:] = inp.B_vv
    eri = np.einsum("Qpq,Qrs->pqrs", B, B)
    u = 2.0 * np.einsum("pqii->pq", eri[:, :, :o, :o]) \
        - np.einsum("piiq->pq", eri[:, :o, :o, :])

    def apply_WN(x):
        y = [[E[r][s] @ x for s in range(n)] for r in range(n)]
        out = np.zeros_like(x)
        for p in range(n):
            for q in range(n):
                z = np.zeros_like(x)
                for r in range(n):
                    for s in range(n):
                        z += eri[p, q, r, s] * y[r][s]
                out += 0.5 * (E[p][q] @ z)
                # - 1/2 sum_s (pq|qs') ... : -1/2 sum_{r=q} (pq|q s) E_ps
        for p in range(n):
            for s in range(n):
                c = 0.5 * sum(eri[p, q, q, s] for q in range(n)) + u[p, s]
                out -= c * y[p][s]
        return out

    # HF determinant: spin orbitals 0..2o-1 occupied; index bit for orbital s is 2^(nso-1-s)
    idx0 = sum(1 << (nso - 1 - s) for s in range(2 * o))
    hf = np.zeros(dim)
    hf[idx0] = 1.0
    eps = np.concatenate([inp.eps_occ, inp.eps_vir])
    return E, apply_WN, hf, eps, nso


def _resolvent(o, eps, nso, rank):
    """diag(1/D) on the determinants with `rank` holes and `rank` particles, D = sum eps_holes - sum eps_particles."""
    dim = 1 << nso
    r = np.zeros(dim)
    for d in range(dim):
        holes, parts, D = 0, 0, 0.0
        for s in range(nso):
            occd = (d >> (nso - 1 - s)) & 1
            p = s // 2
            if p < o and not occd:
                holes += 1
                D += eps[p]
            elif p >= o and occd:
                parts += 1
                D -= eps[p]
        if holes == rank and parts == rank:
            r[d] = 1.0 / D
    return r


def first_principles_mp2(inp):
    """Second-order Rayleigh-Schroedinger energy E2 = <0| W_N R W_N |0> of the model Hamiltonian, R the
    resolvent of H0 on singly and doubly excited determinants.  Uses no index formula of PAPER.md Eq. (1).
    Returns (E2_doubles, E2_singles); the singles part vanishes because W_N is normal ordered w.r.t. the
    HF mean field (Brillouin).  Feasible for o+v <= 7."""
    o = inp.nocc
    E, apply_WN, hf, eps, nso = _model(inp)
    psi = apply_WN(hf)
    r2 = _resolvent(o, eps, nso, 2)
    r1 = _resolvent(o, eps, nso, 1)
    return float(psi @ (r2 * psi)), float(psi @ (r1 * psi))


def first_principles_t(inp, with_fock=False):
    """Return (E4, E5) — or (E4, E5, EF) with `with_fock` — for a TInputs; feasible for o+v <= 7."""
    o, v = inp.nocc, inp.nvir
    E, apply_WN, hf, eps, nso = _model(inp)
    dim = 1 << nso

    t1v = np.zeros(dim)
    for i in range(o):
        for aa in range(v):
            t1v += inp.t1[i, aa] * (E[o + aa][i] @ hf)
    t2v = np.zeros(dim)
    for j in range(o):
        for b in range(v):
            xb = E[o + b][j] @ hf
            for i in range(o):
                for aa in range(v):
                    t2v += 0.5 * inp.t2[i, j, aa, b] * (E[o + aa][i] @ xb)

    psi = apply_WN(t2v)
    phi = apply_WN(t1v)

    # R3 on determinants
    r3 = _resolvent(o, eps, nso, 3)
    e4, e5 = float(psi @ (r3 * psi)), float(phi @ (r3 * psi))
    if not with_fock:
        return e4, e5
    chi = np.zeros(dim)
    for i in range(o):
        for aa in range(v):
            chi += inp.f_ov[i, aa] * ((E[o + aa][i] + E[i][o + aa]) @ t2v)
    return e4, e5, float(chi @ (r3 * psi))
