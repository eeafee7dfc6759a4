"""T0b literal nested loops -- TEST INFRASTRUCTURE, not a product path.

Every term of Omega[i,a,j,b] written as explicit Python loops over every summation
index, with no einsum, no BLAS and no intermediates (O(N^6) for the terms linear in
t, O(N^8) for the quadratic ones).  Guards the index strings of oracle/dense.py and
the wiring of the two ERI sets (reading R6: THC <.|.> in Eqs.32, 33, 35, Cholesky
(.|.) everywhere else).  Only for miniature shapes, (o, v) <= (2, 3) or so.

t is t[i,a,j,b] = t_ij^ab;  g(p,q,r,s) are chemists' ERIs accessed through small
closures so that the formulas below read exactly like PAPER.md Eqs.28-41.
"""
from __future__ import annotations

import itertools
import numpy as np


def omega_terms_naive(t, B_oo, B_ov, B_vv, thc, eps_o, eps_v):
    NL, o, v = B_ov.shape
    O, Vr = range(o), range(v)

    def T(i, j, a, b):            # t_ij^ab
        return t[i, a, j, b]

    def U(i, j, a, b):            # 2 t_ij^ab - t_ij^ba
        return 2.0 * t[i, a, j, b] - t[i, b, j, a]

    def ovov(i, a, j, b):         # (ia|jb)
        return sum(B_ov[L, i, a] * B_ov[L, j, b] for L in range(NL))

    def oooo(i, j, k, l):         # (ij|kl)
        return sum(B_oo[L, i, j] * B_oo[L, k, l] for L in range(NL))

    def oovv(i, j, a, b):         # (ij|ab)
        return sum(B_oo[L, i, j] * B_vv[L, a, b] for L in range(NL))

    def vvvv(a, b, c, d):         # (ab|cd)
        return sum(B_vv[L, a, b] * B_vv[L, c, d] for L in range(NL))

    def X(i, a, j, b):            # <ia|jb>  (THC set)
        return thc[i, a, j, b]

    # Eq.39 / Eq.40
    xi_oo = np.zeros((o, o))
    for k, j in itertools.product(O, O):
        xi_oo[k, j] = sum(T(j, m, d, e) * (2.0 * ovov(m, e, k, d) - ovov(m, d, k, e))
                          for m in O for d in Vr for e in Vr)
    xi_vv = np.zeros((v, v))
    for b, c in itertools.product(Vr, Vr):
        xi_vv[b, c] = -sum(T(l, m, d, b) * (2.0 * ovov(l, d, m, c) - ovov(l, c, m, d))
                           for l in O for m in O for d in Vr)

    def Foo(k, j):
        return (eps_o[k] if k == j else 0.0) + xi_oo[k, j]

    def Fvv(b, c):
        return (eps_v[b] if b == c else 0.0) + xi_vv[b, c]

    out = {k: np.zeros((o, v, o, v)) for k in ("s1", "s2", "s3", "s6", "s7", "s9")}
    for i, a, j, b in itertools.product(O, Vr, O, Vr):
        # Eq.29
        out["s2"][i, a, j, b] = (ovov(i, a, j, b)
                                 + sum(U(i, k, a, c) * ovov(j, b, k, c) for k in O for c in Vr)
                                 + sum(U(j, k, b, c) * ovov(i, a, k, c) for k in O for c in Vr))
        # Eq.28
        out["s1"][i, a, j, b] = (sum(T(i, j, c, d) * vvvv(a, c, b, d) for c in Vr for d in Vr)
                                 + sum(T(k, l, a, b) * oooo(k, i, l, j) for k in O for l in O)
                                 - sum(T(i, l, c, b) * oovv(l, j, a, c) for l in O for c in Vr)
                                 - sum(T(k, j, a, d) * oovv(k, i, b, d) for k in O for d in Vr))
        # Eq.31
        out["s3"][i, a, j, b] = -sum(T(i, k, a, c) * oovv(k, j, b, c) + T(j, k, b, c) * oovv(k, i, a, c)
                                     for k in O for c in Vr)
        # Eq.32 + Eq.33
        out["s6"][i, a, j, b] = sum(T(i, j, c, d) * T(k, l, a, b) * X(k, c, l, d)
                                    + T(i, k, c, b) * T(l, j, a, d) * X(l, c, k, d)
                                    for k in O for l in O for c in Vr for d in Vr)
        # Eq.35 with prefactor 1/2 and (2t - t) in both brackets (readings R2, R3)
        out["s7"][i, a, j, b] = 0.5 * sum(
            U(i, k, a, c) * (2.0 * X(k, c, l, d) - X(k, d, l, c)) * U(j, l, b, d)
            + T(i, k, c, a) * X(k, d, l, c) * T(j, l, d, b)
            for k in O for l in O for c in Vr for d in Vr)
        # Eq.41 in the symmetric form of Alg.9 (reading R4)
        out["s9"][i, a, j, b] = (sum(T(i, j, a, c) * Fvv(b, c) for c in Vr)
                                 + sum(T(i, j, c, b) * Fvv(a, c) for c in Vr)
                                 - sum(T(i, k, a, b) * Foo(k, j) for k in O)
                                 - sum(T(k, j, a, b) * Foo(k, i) for k in O))
    out["xi_oo"], out["xi_vv"] = xi_oo, xi_vv
    return out


def project_naive(Xo, Xv, omega):
    o, NP = Xo.shape
    v = Xv.shape[0]
    R = np.zeros((NP, NP))
    for P in range(NP):
        for Q in range(NP):
            R[P, Q] = sum(Xo[i, P] * Xv[a, P] * omega[i, a, j, b] * Xo[j, Q] * Xv[b, Q]
                          for i in range(o) for a in range(v) for j in range(o) for b in range(v))
    return R


def expand_t_naive(Xo, Xv, Z):
    o, NP = Xo.shape
    v = Xv.shape[0]
    t = np.zeros((o, v, o, v))
    for i, a, j, b in itertools.product(range(o), range(v), range(o), range(v)):
        t[i, a, j, b] = sum(Xo[i, P] * Xv[a, P] * Z[P, Q] * Xo[j, Q] * Xv[b, Q]
                            for P in range(NP) for Q in range(NP))
    return t
