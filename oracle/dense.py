"""T1 dense oracle (oracle of record) -- TEST INFRASTRUCTURE, not a product path.

Computes, in plain numpy float64 and straight from the definitions,

    R_PQ = sum_ijab Xo[i,P] Xv[a,P] Omega[i,a,j,b] Xo[j,Q] Xv[b,Q]      (north_star; Eq.6 l.82
                                                                          with U^P_ia -> Xo_iP Xv_aP, Eq.23 l.193)
    E    = sum_ijab (2 t_ij^ab - t_ij^ba) (ia|jb)                        ("same as usual in CCSD", l.80)

where t is expanded densely from its THC factors (Eq.23 l.193), the Cholesky ERIs
are rebuilt as explicit 4-index arrays (Eq.24 l.199) and the THC ERIs likewise
(Eq.17 l.141).  Omega is the closed-shell CCSD doubles residual at t1 = 0 written
as the sum of the paper's dense equations 28, 29, 31, 32+33 (=34), 35, 41 with the
readings R1-R7 of DESIGN.md section 3 (Eq.35 prefactor 1/2 and (2t - t) in both
brackets; Eq.41 in the ia<->jb symmetric form Alg.9 computes; THC ERIs exactly in
Eqs.32, 33, 35; Cholesky ERIs everywhere else, including xi and the energy).

No blocking, no fusion, no reuse of the factorised identities the CUDA path uses:
`o_PQ`, `v_PQ`, Hadamard tricks etc. never appear here.

Array convention: every 4-index amplitude/residual is stored [i, a, j, b], i.e.
t[i,a,j,b] = t_ij^ab;  ERIs are stored in chemists' order, e.g. ovov[i,a,j,b] = (ia|jb).

Pins: tests/test_oracle_*.py check this file against the determinant-space brute
force (oracle/bruteforce.py), literal loops (oracle/naive.py), the paper's
factorised algorithms transcribed in tests/paper_algorithms.py, closed forms and
invariants.
"""
from __future__ import annotations

import numpy as np

TERMS = ("s1", "s2", "s3", "s6", "s7", "s9")


def expand_t(Xo, Xv, Z):
    """t[i,a,j,b] = sum_PQ Xo[i,P] Xv[a,P] Z[P,Q] Xo[j,Q] Xv[b,Q]   (Eq.23 l.193)."""
    U = np.einsum("iP,aP->iaP", Xo, Xv, optimize=True)
    return np.einsum("iaP,PQ,jbQ->iajb", U, Z, U, optimize=True)


def cd_eris(B_oo, B_ov, B_vv):
    """Explicit Cholesky ERIs (pq|rs) = sum_L B^L_pq B^L_rs   (Eq.24 l.199, t1 = 0)."""
    return dict(
        ovov=np.einsum("Lia,Ljb->iajb", B_ov, B_ov, optimize=True),
        oooo=np.einsum("Lij,Lkl->ijkl", B_oo, B_oo, optimize=True),
        oovv=np.einsum("Lij,Lab->ijab", B_oo, B_vv, optimize=True),
        vvvv=np.einsum("Lab,Lcd->abcd", B_vv, B_vv, optimize=True),
    )


def thc_ovov(Yo, Yv, V):
    """<ia|jb> = sum_IJ Yo[i,I] Yv[a,I] V[I,J] Yo[j,J] Yv[b,J]   (Eq.17 l.141)."""
    W = np.einsum("iI,aI->iaI", Yo, Yv, optimize=True)
    return np.einsum("iaI,IJ,jbJ->iajb", W, V, W, optimize=True)


def xi_intermediates(t, ovov):
    """xi_kj (Eq.39 l.280) and xi_bc (Eq.40 l.283), Cholesky ERIs (Alg.8 uses l_ia, l.796-798).

    xi_oo[k,j] = sum_mde t_jm^de [2 (me|kd) - (md|ke)]
    xi_vv[b,c] = - sum_lmd t_lm^db [2 (ld|mc) - (lc|md)]
    """
    # t_jm^de = t[j,d,m,e];  (me|kd) = ovov[m,e,k,d];  (md|ke) = ovov[m,d,k,e]
    xi_oo = 2.0 * np.einsum("jdme,mekd->kj", t, ovov, optimize=True) - np.einsum("jdme,mdke->kj", t, ovov, optimize=True)
    # t_lm^db = t[l,d,m,b];  (ld|mc) = ovov[l,d,m,c];  (lc|md) = ovov[l,c,m,d]
    xi_vv = -(2.0 * np.einsum("ldmb,ldmc->bc", t, ovov, optimize=True) - np.einsum("ldmb,lcmd->bc", t, ovov, optimize=True))
    return xi_oo, xi_vv


def omega_terms(t, cd, thc, eps_o, eps_v):
    """The six groups of Omega[i,a,j,b], named after the algorithm that evaluates them.

    s2: Eq.29 l.224     s1: Eq.28 l.217     s3: Eq.31 l.235
    s6: Eqs.32+33 l.244-247 (THC ERIs)      s7: Eq.35 l.261 corrected (THC ERIs)
    s9: Eq.41 l.290 in Alg.9's symmetric form, F' = diag(eps) + xi
    """
    ovov, oooo, oovv, vvvv = cd["ovov"], cd["oooo"], cd["oovv"], cd["vvvv"]
    u = 2.0 * t - t.transpose(0, 3, 2, 1)          # u_ik^ac = 2 t_ik^ac - t_ik^ca, stored [i,a,k,c]
    out = {}

    # Eq.29: (ia|jb) + sum_kc u_ik^ac (jb|kc) + sum_kc u_jk^bc (ia|kc)
    out["s2"] = (ovov
                 + np.einsum("iakc,jbkc->iajb", u, ovov, optimize=True)
                 + np.einsum("jbkc,iakc->iajb", u, ovov, optimize=True))

    # Eq.28: sum_cd t_ij^cd (ac|bd) + sum_kl t_kl^ab (ki|lj)
    #        - sum_lc t_il^cb (ac|lj) - sum_kd t_kj^ad (ki|bd)
    out["s1"] = (np.einsum("icjd,acbd->iajb", t, vvvv, optimize=True)
                 + np.einsum("kalb,kilj->iajb", t, oooo, optimize=True)
                 - np.einsum("iclb,ljac->iajb", t, oovv, optimize=True)
                 - np.einsum("kajd,kibd->iajb", t, oovv, optimize=True))

    # Eq.31: - sum_kc [ t_ik^ac (kj|bc) + t_jk^bc (ki|ac) ]
    out["s3"] = -(np.einsum("iakc,kjbc->iajb", t, oovv, optimize=True)
                  + np.einsum("jbkc,kiac->iajb", t, oovv, optimize=True))

    # Eq.32: sum_klcd t_ij^cd t_kl^ab <kc|ld> ;  Eq.33: sum_klcd t_ik^cb t_lj^ad <lc|kd>
    x32 = np.einsum("icjd,kcld->ijkl", t, thc, optimize=True)
    s32 = np.einsum("ijkl,kalb->iajb", x32, t, optimize=True)
    x33 = np.einsum("ickb,lckd->ibld", t, thc, optimize=True)      # sum_kc t_ik^cb <lc|kd>
    s33 = np.einsum("ibld,lajd->iajb", x33, t, optimize=True)      # sum_ld (..) t_lj^ad
    out["s6"] = s32 + s33

    # Eq.35 (corrected): 1/2 sum_klcd [ u_ik^ac (2<kc|ld> - <kd|lc>) u_jl^bd + t_ik^ca <kd|lc> t_jl^db ]
    w = 2.0 * thc - thc.transpose(0, 3, 2, 1)       # w[k,c,l,d] = 2<kc|ld> - <kd|lc>
    y1 = np.einsum("iakc,kcld->iald", u, w, optimize=True)
    p1 = np.einsum("iald,jbld->iajb", y1, u, optimize=True)
    tx = t.transpose(0, 3, 2, 1)                    # tx[i,a,k,c] = t_ik^ca
    thx = thc.transpose(0, 3, 2, 1)                 # thx[k,c,l,d] = <kd|lc>
    y2 = np.einsum("iakc,kcld->iald", tx, thx, optimize=True)
    p2 = np.einsum("iald,jbld->iajb", y2, tx, optimize=True)
    out["s7"] = 0.5 * (p1 + p2)

    # Eq.41 (Alg.9 form): sum_c t_ij^ac F'_bc + sum_c t_ij^cb F'_ac - sum_k t_ik^ab F'_kj - sum_k t_kj^ab F'_ki
    xi_oo, xi_vv = xi_intermediates(t, ovov)
    Foo = np.diag(eps_o) + xi_oo                    # F'[k,j]
    Fvv = np.diag(eps_v) + xi_vv                    # F'[b,c]
    out["s9"] = (np.einsum("iajc,bc->iajb", t, Fvv, optimize=True)
                 + np.einsum("icjb,ac->iajb", t, Fvv, optimize=True)
                 - np.einsum("iakb,kj->iajb", t, Foo, optimize=True)
                 - np.einsum("kajb,ki->iajb", t, Foo, optimize=True))
    out["xi_oo"], out["xi_vv"] = xi_oo, xi_vv
    return out


def project(Xo, Xv, omega):
    """R_PQ = sum_ijab Xo[i,P] Xv[a,P] Omega[i,a,j,b] Xo[j,Q] Xv[b,Q]."""
    U = np.einsum("iP,aP->iaP", Xo, Xv, optimize=True)
    return np.einsum("iaP,iajb,jbQ->PQ", U, omega, U, optimize=True)


def energy_from(t, ovov):
    """E = sum_ijab (2 t_ij^ab - t_ij^ba)(ia|jb), Cholesky ERIs (reading R7)."""
    u = 2.0 * t - t.transpose(0, 3, 2, 1)
    return float(np.einsum("iajb,iajb->", u, ovov, optimize=True))


def residual_and_energy(Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, thc_from_cd=False):
    """Full oracle evaluation.

    Returns a dict with R (total), one projected matrix per term (TERMS), xi_oo,
    xi_vv, E, and the dense Omega terms under "omega" (for the brute-force pins).
    `thc_from_cd=True` replaces the THC ERI set by the Cholesky one (only used to
    compare against the determinant-space brute force, which knows one Hamiltonian).
    """
    o = Xo.shape[0]
    eps_o, eps_v = eps[:o], eps[o:]
    t = expand_t(Xo, Xv, Z)
    cd = cd_eris(B_oo, B_ov, B_vv)
    thc = cd["ovov"] if thc_from_cd else thc_ovov(Y[:o], Y[o:], V)
    om = omega_terms(t, cd, thc, eps_o, eps_v)
    res = {"omega": {k: om[k] for k in TERMS}, "xi_oo": om["xi_oo"], "xi_vv": om["xi_vv"]}
    total = np.zeros((Xo.shape[1], Xo.shape[1]))
    for k in TERMS:
        res[k] = project(Xo, Xv, om[k])
        total += res[k]
    res["R"] = total
    res["E"] = energy_from(t, cd["ovov"])
    res["t"] = t
    return res
