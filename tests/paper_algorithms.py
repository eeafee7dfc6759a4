"""PAPER.md Algorithms 1, 2, 3, 6, 7, 8 (lines 5-10) and 9 transcribed line by line in numpy.

Test helper: the north_star's "identity between factorized and dense contractions" pin
for oracle/dense.py.  Each function follows the listing in PAPER.md (l.480-843) in the
paper's own order and notation (y = amplitude THC factors, T = core matrix, x / z = ERI
THC factors, l_ij / l_ia / l_ab = one Cholesky vector in the MO basis, t1 = 0), with the
garbled lines read as in DESIGN.md section 3 (R2, R3, R10, R11, R12).  It shares nothing
with the CUDA path (which fuses, reorders and blocks these steps) and nothing with
oracle/dense.py (which never forms o^{XY}, v^{XY} or any Hadamard intermediate).
"""
import numpy as np


def alg1(yo, yv, T, l_oo, l_vv):
    """Algorithm 1 (l.480-530): ladder terms linear in T2, Eq.28."""
    o_ = yo.T @ yo                                     # 1: o^{XY}
    v_ = yv.T @ yv                                     # 2: v^{XY}
    sigma = np.zeros_like(T)
    for A in range(l_oo.shape[0]):                     # 3
        lij, lab = l_oo[A], l_vv[A]                    # 4,5,9 (already MO basis, t1 = 0)
        Abar = np.einsum("kX,ki->iX", yo, lij)         # 6:  Abar_i^X = sum_k y_k^X l_ki
        Bbar = np.einsum("iX,iY->XY", Abar, yo)        # 7
        Cbar = v_ * Bbar                               # 8
        Atil = np.einsum("aX,ac->cX", yv, lab)         # 10
        Btil = np.einsum("cX,cY->XY", Atil, yv)        # 11
        Ctil = o_ * Btil                               # 12
        C = Cbar - Ctil                                # 13
        D = C @ T                                      # 14: D^{XY'} = sum_Y C^{XY} T^{YY'}
        sigma += D @ C.T                               # 15: sigma^{XX'} += sum_Y' D^{XY'} C^{X'Y'}
    return sigma


def alg2(yo, yv, T, l_ov):
    """Algorithm 2 (l.532-567): bare ERI + ring terms linear in T2, Eq.29."""
    sigma = np.zeros_like(T)
    for A in range(l_ov.shape[0]):
        lia = l_ov[A]                                  # 3 (l_ai = l_ia^T when t1 = 0)
        Abar = np.einsum("aX,iX,ia->X", yv, yo, lia)   # 4
        Atil = np.einsum("iX,aX,ia->X", yo, yv, lia)   # 5
        Btil = T @ Atil                                # 6
        Ctil = np.einsum("iY,aY,Y->ia", yo, yv, Btil)  # 7
        Dtil = np.einsum("iX,aX,ia->X", yo, yv, Ctil)  # 8
        E = np.einsum("cY,kZ,kc->YZ", yv, yo, lia)     # 9:  E^{YY'} = sum_kc y_c^Y y_k^{Y'} l_kc
        F = T * E                                      # 10
        G = np.einsum("iY,aZ,YZ->ia", yo, yv, F)       # 11: G_ia = sum_{YY'} y_i^Y y_a^{Y'} F^{YY'}
        H = np.einsum("iX,aX,ia->X", yo, yv, G)        # 12
        sigma += (np.outer(Abar, Abar) + 2 * np.outer(Dtil, Abar) + 2 * np.outer(Abar, Dtil)
                  - np.outer(H, Abar) - np.outer(Abar, H))          # 13
    return sigma


def alg3(yo, yv, T, l_oo, l_vv):
    """Algorithm 3 (l.569-606): remaining Omega^C terms linear in T2, Eq.31."""
    C = np.zeros_like(T)
    for A in range(l_oo.shape[0]):
        Amat = np.einsum("bX,cY,bc->XY", yv, yv, l_vv[A])   # 5
        Bmat = np.einsum("jX,kY,kj->XY", yo, yo, l_oo[A])   # 6
        C += Amat * Bmat                                    # 7
    o_ = yo.T @ yo                                          # 9
    v_ = yv.T @ yv                                          # 10
    D = (o_ * v_) @ T                                       # 11
    return -D @ C.T - C @ D.T                               # 12


def alg6(yo, yv, T, xo, xv, z):
    """Algorithm 6 (l.682-730): O(N^4) evaluation of Eqs.32+33 with THC ERIs (reading R10)."""
    NX = z.shape[0]
    NP = T.shape[0]
    A = np.einsum("iY,aY,XY->iaX", yo, yv, T)          # 1: A_ia^X
    Bt = np.einsum("iJ,aJ,IJ->iaI", xo, xv, z)         # 2: B_ia^I
    C = np.einsum("aX,iaY->iXY", yv, A)                # 4: C_i^{XY}
    D = np.einsum("iX,iaY->aXY", yo, A)                # 5: D_a^{XY}
    H = np.zeros((NP, NP, NP))
    for I in range(NX):                                # 6 (missing line: "for I do")
        b = Bt[:, :, I]                                # 7
        E = np.einsum("iXY,i->XY", C, xo[:, I])        # 8
        F = np.einsum("aXZ,a->XZ", D, xv[:, I])        # 9
        G = np.einsum("iY,aZ,ia->YZ", yo, yv, b)       # 10
        H += (E[:, :, None] * F[:, None, :] + E[:, None, :] * F[:, :, None]) * G[None, :, :]  # 11
    sigma = np.zeros_like(T)
    for X in range(NP):                                # 13
        Iia = np.einsum("iZ,aY,YZ->ia", yo, yv, H[X])  # 14
        sigma[X, :] = np.einsum("iY,aY,ia->Y", yo, yv, Iia)   # 15: sigma^{XX'}
    return sigma


def alg7(yo, yv, T, xo, xv, z):
    """Algorithm 7 (l.732-773): ring-type T2^2 terms, Eqs.35-37, prefactor 1/2 (R2, R11, R12)."""
    NP = T.shape[0]
    o_ = yo.T @ yo                                     # 1
    v_ = yv.T @ yv                                     # 2
    A = (o_ * v_) @ T.T                                # 3: A^{XY} = sum_Z o^{XZ} v^{XZ} T^{YZ}
    R = 2 * np.einsum("iY,aY,XY->Xia", yo, yv, A)      # 4
    S = np.zeros_like(R)
    for X in range(NP):                                # 5
        Bm = v_[X][:, None] * o_[X][None, :] * T       # 6: B^{YZ} = v^{XY} o^{XZ} T^{YZ}
        S[X] = -np.einsum("iY,aZ,YZ->ia", yo, yv, Bm)  # 7: defines S and adds it to R (R12)
        R[X] += S[X]
    C = np.einsum("iI,aI,Xia->XI", xo, xv, R)          # 9
    D = C @ z.T                                        # 10: D^{XI} = sum_J C^{XJ} z^{IJ}
    G = np.zeros_like(R)
    Gt = np.zeros_like(R)
    for X in range(NP):                                # 12
        E = np.einsum("iI,aJ,ia->IJ", xo, xv, R[X])    # 13
        F = E * z                                      # 14
        G[X] = np.einsum("jJ,bI,IJ->jb", xo, xv, F)    # 15
        Et = np.einsum("iI,aJ,ia->IJ", xo, xv, S[X])   # 17
        Ft = Et * z                                    # 18
        Gt[X] = np.einsum("jJ,bI,IJ->jb", xo, xv, Ft)  # 19
    return 0.5 * (2 * C @ D.T - np.einsum("Xia,Yia->XY", G, R)
                  + np.einsum("Xia,Yia->XY", Gt, S))   # 22 with 1/2 (R2)


def alg8_xi(yo, yv, T, l_ov):
    """Algorithm 8 lines 5-10 (l.777-809): xi_ij (Eq.39) and xi_ab (Eq.40)."""
    o, v = yo.shape[0], yv.shape[0]
    xi_oo, xi_vv = np.zeros((o, o)), np.zeros((v, v))
    for A in range(l_ov.shape[0]):
        lia = l_ov[A]
        Avec = np.einsum("iX,aX,ia->X", yo, yv, lia)          # 5
        Bm = np.einsum("iX,aY,ia->XY", yo, yv, lia)           # 6
        Cm = 2 * np.diag(T @ Avec) - Bm * T                   # 7
        Dia = np.einsum("iY,aX,XY->ia", yo, yv, Cm)           # 8
        xi_oo += np.einsum("ia,ja->ij", lia, Dia)             # 9
        xi_vv -= np.einsum("ia,ib->ab", Dia, lia)             # 10
    return xi_oo, xi_vv


def alg9(yo, yv, T, F_oo, F_vv):
    """Algorithm 9 (l.811-843): Omega^E; F_oo[j,i] = F_ji + xi_ji, F_vv[a,b] = F_ab + xi_ab."""
    o_ = yo.T @ yo                                     # 1
    v_ = yv.T @ yv                                     # 2
    A = o_ * v_                                        # 3
    B = A @ T                                          # 4
    C = np.einsum("ji,jX->iX", F_oo, yo)               # 5: C_i^X = sum_j (F_ji + xi_ji) y_j^X
    D = np.einsum("ab,bX->aX", F_vv, yv)               # 6
    ot = np.einsum("iX,iY->XY", yo, C)                 # 7
    vt = np.einsum("aX,aY->XY", yv, D)                 # 8
    E = o_ * vt - ot * v_                              # 9
    return E @ B.T + B @ E.T                           # 10
