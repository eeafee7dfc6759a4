"""Rank-reduced (RR) working variables -- TEST INFRASTRUCTURE, not a product path.

PAPER.md Eqs.13-14 (l.116-120) and Eq.22 (l.178-181): with the orthogonalised CP factor tau~[P, W] the projectors are
U~^P_ia = sum_W y_i^W y_a^W tau~[P, W] (Eq.14), the amplitudes t_ij^ab = sum_PQ U~^P_ia T^{PQ} U~^Q_jb (Eq.22, "we
recommend the former", l.181) and the amplitude equations are projected with the same U~ (Eq.6 l.82):

    R^RR_PQ = sum_ijab U~^P_ia Omega_ijab U~^Q_jb .

This file writes exactly that out with dense arrays: U~ is formed as a 3-index array, t and the projection use it
directly.  The THC-auxiliary-basis core Z = tau~^T T tau~ and the identity R^RR = tau~ sigma tau~^T that the CUDA path
uses never appear here.  Omega is dense.omega_terms (the oracle of record, pinned by the determinant-space brute force).

symmetric_orthogonalizer() is Eqs.10-13: S = tau (o .* v) tau^T, tau~ = S^{-1/2} tau; the input generators of the tests
use it to draw a tau~ whose projectors are semi-unitary (Eq.12), which tests/test_oracle_rr.py checks.
"""
from __future__ import annotations

import numpy as np

from . import dense


def projectors(Xo, Xv, tau):
    """U~[i, a, P] = sum_W Xo[i,W] Xv[a,W] tau[P,W]   (Eq.14 l.120)."""
    return np.einsum("iW,aW,PW->iaP", Xo, Xv, tau, optimize=True)


def symmetric_orthogonalizer(Xo, Xv, tau):
    """tau~ = S^{-1/2} tau with S^{PQ} = sum_ia U^P_ia U^Q_ia   (Eqs.10, 11, 13 l.103-116)."""
    U = projectors(Xo, Xv, tau)
    S = np.einsum("iaP,iaQ->PQ", U, U, optimize=True)
    w, Q = np.linalg.eigh(S)
    return (Q * (1.0 / np.sqrt(w))) @ Q.T @ tau


def rr_residual_and_energy(Xo, Xv, tau, T, B_ov, B_oo, B_vv, Y, V, eps):
    """dict(R_rr [NR, NR], E, t) for amplitudes t = U~ T U~^T (Eq.22) and the projection of Eq.6 with U~."""
    o = Xo.shape[0]
    U = projectors(Xo, Xv, tau)
    t = np.einsum("iaP,PQ,jbQ->iajb", U, T, U, optimize=True)
    cd = dense.cd_eris(B_oo, B_ov, B_vv)
    thc = dense.thc_ovov(Y[:o], Y[o:], V)
    om = dense.omega_terms(t, cd, thc, eps[:o], eps[o:])
    omega = sum(om[k] for k in dense.TERMS)
    return dict(R_rr=np.einsum("iaP,iajb,jbQ->PQ", U, omega, U, optimize=True), E=dense.energy_from(t, cd["ovov"]), t=t)
