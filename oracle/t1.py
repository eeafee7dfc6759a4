"""T1-dressed closed-shell CCSD residuals (singles and doubles), dense -- TEST INFRASTRUCTURE, not a product path.

PAPER.md l.197-213: "The use of a T1 transformation of the Hamiltonian is utilized throughout"; the t1 amplitudes enter
only through the dressed MO coefficients (Eqs.25-26), i.e. in the MO basis (C = 1) through

    Xp[r, a] = delta_ra - sum_i t_i^a delta_ri          (C^p: virtual columns get -t_i^a in row i)
    Xh[s, i] = delta_si + sum_a t_i^a delta_sa          (C^h: occupied columns get +t_i^a in row a)
    B^_pq    = sum_rs Xp[r, p] B_rs Xh[s, q]            (Eq.27 l.209; only 2-fold bra-ket symmetry remains, l.211)

and every "hatted" integral is (pq|rs)^ = sum_L B^_pq B^_rs (Eq.24 l.199).  The one-electron part follows the same
transformation, h^ = Xp^T h Xh, with h fixed by the bare Fock matrix being diag(eps) (reading R1/R8: canonical orbitals),
and the dressed inactive Fock matrix is F^_pq = h^_pq + sum_k [2 (pq|kk)^ - (pk|kq)^].

Residuals (dense arrays, equations as printed, with the readings of DESIGN.md section 3 for Eqs.35 and 41):

  doubles   Omega_ijab = Eq.29 + Eq.28 + Eq.31 (hatted Cholesky ERIs) + Eqs.32, 33, 35 (THC <ov|ov>, untouched by the
            dressing because B^_ia = B_ia) + Eq.41 with F^ + xi                              -> terms s2 s1 s3 s6 s7 s9
  singles   sigma_ia   = Eq.38 (Omega G, H) + Eq.42 (Omega I, J)                              l.277, l.295

Pinned by tests/test_oracle_t1.py: determinant-space <mu| exp(-T1-T2) H exp(T1+T2) |Phi0> (oracle/bruteforce.py, no CC
formula), reduction to oracle/dense.py at t1 = 0, and the dressing identities.
"""
from __future__ import annotations

import numpy as np

from . import dense

TERMS = dense.TERMS


def full_B(B_oo, B_ov, B_vv):
    """Bare Cholesky vectors over all o+v orbitals, [NL, n, n] (vo block = ov^T)."""
    NL, o, v = B_ov.shape
    B = np.zeros((NL, o + v, o + v))
    B[:, :o, :o], B[:, :o, o:], B[:, o:, :o], B[:, o:, o:] = B_oo, B_ov, B_ov.transpose(0, 2, 1), B_vv
    return B


def dressing_matrices(t1):
    """Xp, Xh of Eqs.25-26 in the MO basis."""
    o, v = t1.shape
    Xp, Xh = np.eye(o + v), np.eye(o + v)
    Xp[:o, o:] = -t1
    Xh[o:, :o] = t1.T
    return Xp, Xh


def dress(B, t1):
    """B^[L, p, q] = sum_rs Xp[r, p] B[L, r, s] Xh[s, q]   (Eq.27 l.209)."""
    Xp, Xh = dressing_matrices(t1)
    return np.einsum("rp,Lrs,sq->Lpq", Xp, B, Xh, optimize=True)


def dressed_fock(B, Bh, t1, eps):
    """F^[p, q] = h^_pq + sum_k [2 (pq|kk)^ - (pk|kq)^],  h^ = Xp^T h Xh,  h = diag(eps) - sum_k [2 (pq|kk) - (pk|kq)]."""
    o = t1.shape[0]
    Xp, Xh = dressing_matrices(t1)

    def g(Bx):
        return 2.0 * np.einsum("Lpq,Lkk->pq", Bx, Bx[:, :o, :o], optimize=True) - np.einsum("Lpk,Lkq->pq", Bx[:, :, :o], Bx[:, :o, :], optimize=True)
    h = np.diag(np.asarray(eps, dtype=float)) - g(B)
    return Xp.T @ h @ Xh + g(Bh)


def residuals(t1, t, B_oo, B_ov, B_vv, thc, eps):
    """dict: omega terms s1..s9 [i,a,j,b], sigma_G_H, sigma_I_J, sigma [i,a], xi_oo, xi_vv, F (dressed Fock, [n, n])."""
    o, v = t1.shape
    B = full_B(B_oo, B_ov, B_vv)
    Bh = dress(B, t1)
    O, Vv = slice(0, o), slice(o, o + v)
    blk = {"o": O, "v": Vv}

    def eri(s):              # (pq|rs)^ for a block string such as "vovo"
        return np.einsum("Lpq,Lrs->pqrs", Bh[:, blk[s[0]], blk[s[1]]], Bh[:, blk[s[2]], blk[s[3]]], optimize=True)
    F = dressed_fock(B, Bh, t1, eps)
    u = 2.0 * t - t.transpose(0, 3, 2, 1)                 # u[i,a,k,c] = 2 t_ik^ac - t_ik^ca
    ovov = eri("ovov")                                     # = bare (ia|jb): B^_ia = B_ia
    out = {}
    # Eq.29 l.224: (ai|bj)^ + sum_kc u_ik^ac (bj|kc)^ + sum_kc u_jk^bc (ai|kc)^
    vovo, voov = eri("vovo"), eri("voov")
    out["s2"] = (vovo.transpose(1, 0, 3, 2)
                 + np.einsum("iakc,bjkc->iajb", u, voov, optimize=True)
                 + np.einsum("jbkc,aikc->iajb", u, voov, optimize=True))
    # Eq.28 l.217: sum_cd t_ij^cd (ac|bd)^ + sum_kl t_kl^ab (ki|lj)^ - sum_lc t_il^cb (ac|lj)^ - sum_kd t_kj^ad (ki|bd)^
    vvvv, oooo, vvoo, oovv = eri("vvvv"), eri("oooo"), eri("vvoo"), eri("oovv")
    out["s1"] = (np.einsum("icjd,acbd->iajb", t, vvvv, optimize=True)
                 + np.einsum("kalb,kilj->iajb", t, oooo, optimize=True)
                 - np.einsum("iclb,aclj->iajb", t, vvoo, optimize=True)
                 - np.einsum("kajd,kibd->iajb", t, oovv, optimize=True))
    # Eq.31 l.235: - sum_kc [ t_ik^ac (kj|bc)^ + t_jk^bc (ki|ac)^ ]
    out["s3"] = -(np.einsum("iakc,kjbc->iajb", t, oovv, optimize=True)
                  + np.einsum("jbkc,kiac->iajb", t, oovv, optimize=True))
    # Eqs.32, 33, 35 and the xi intermediates use <ov|ov> / (ov|ov) only: unchanged by the dressing; reuse the t1 = 0 code
    base = dense.omega_terms(t, dict(ovov=ovov, oooo=oooo, oovv=oovv, vvvv=vvvv), thc, np.zeros(o), np.zeros(v))
    out["s6"], out["s7"] = base["s6"], base["s7"]
    xi_oo, xi_vv = base["xi_oo"], base["xi_vv"]
    # Eq.41 l.290 (Alg.9 form) with F' = F^ + xi
    Foo, Fvv = F[O, O] + xi_oo, F[Vv, Vv] + xi_vv
    out["s9"] = (np.einsum("iajc,bc->iajb", t, Fvv, optimize=True) + np.einsum("icjb,ac->iajb", t, Fvv, optimize=True)
                 - np.einsum("iakb,kj->iajb", t, Foo, optimize=True) - np.einsum("kajb,ki->iajb", t, Foo, optimize=True))
    # Eq.38 l.277: sum_kcd t_ik^cd [2 (kd|ac)^ - (kc|ad)^] - sum_klc t_kl^ac [2 (lc|ki)^ - (li|kc)^]
    ovvv, ovoo, ooov = eri("ovvv"), eri("ovoo"), eri("ooov")
    out["sigma_G_H"] = (2.0 * np.einsum("ickd,kdac->ia", t, ovvv, optimize=True) - np.einsum("ickd,kcad->ia", t, ovvv, optimize=True)
                        - 2.0 * np.einsum("kalc,lcki->ia", t, ovoo, optimize=True) + np.einsum("kalc,likc->ia", t, ooov, optimize=True))
    # Eq.42 l.295: F^_ai + sum_kc u_ik^ac F^_kc
    out["sigma_I_J"] = F[Vv, O].T + np.einsum("iakc,kc->ia", u, F[O, Vv], optimize=True)
    out["sigma"] = out["sigma_G_H"] + out["sigma_I_J"]
    out["xi_oo"], out["xi_vv"], out["F"] = xi_oo, xi_vv, F
    return out


def residual_and_energy(Xo, Xv, Z, t1, B_ov, B_oo, B_vv, Y, V, eps, thc_from_cd=False):
    """Projected doubles residual per term and in total, the singles residual, and the dense Omega terms."""
    o = Xo.shape[0]
    t = dense.expand_t(Xo, Xv, Z)
    thc = np.einsum("Lia,Ljb->iajb", B_ov, B_ov, optimize=True) if thc_from_cd else dense.thc_ovov(Y[:o], Y[o:], V)
    om = residuals(t1, t, B_oo, B_ov, B_vv, thc, eps)
    res = {"omega": {k: om[k] for k in TERMS}, "sigma": om["sigma"], "sigma_G_H": om["sigma_G_H"], "sigma_I_J": om["sigma_I_J"],
           "xi_oo": om["xi_oo"], "xi_vv": om["xi_vv"], "F": om["F"], "t": t}
    total = np.zeros((Xo.shape[1], Xo.shape[1]))
    for k in TERMS:
        res[k] = dense.project(Xo, Xv, om[k])
        total += res[k]
    res["R"] = total
    return res
