"""MP2 one-particle density matrix from THC-factorised doubles -- TEST INFRASTRUCTURE, not a product path.

PAPER.md Appendix II (l.375-415).  The quantity has a plain definition, Eqs.47-48 (l.379-383):

    D_ij = -2 sum_kab t_ik^ab [2 t_jk^ab - t_jk^ba]                      (47)
    D_ab =  2 sum_ijc t_ij^ac [2 t_ij^bc - t_ji^bc]                      (48)

with the amplitudes of Eq.23 (l.193), t_ij^ab = sum_PQ Xo[i,P] Xv[a,P] Z[P,Q] Xo[j,Q] Xv[b,Q].  The oracle is that
definition written out on the dense 4-index array (O(N^5) work, O(N^4) memory: small cases only).  The O(N^4)
factorisation of Eqs.53-56 that the CUDA path evaluates does not appear here; tests/test_oracle_mp2_density.py pins this
file against literal loops, a closed form, trace / definiteness invariants and a restatement of Eqs.53-56.

Index convention of the dense array: t[i, a, j, b] = t_ij^ab (as oracle/dense.py).
"""
from __future__ import annotations

import numpy as np

from . import dense


def density_from_amplitudes(t):
    """(D_oo [o, o], D_vv [v, v]) of Eqs.47-48 from t[i, a, j, b] = t_ij^ab."""
    # t_jk^ba = t[j, b, k, a];  t_ji^bc = t[j, b, i, c]
    D_oo = -2.0 * (2.0 * np.einsum("iakb,jakb->ij", t, t) - np.einsum("iakb,jbka->ij", t, t))
    D_vv = 2.0 * (2.0 * np.einsum("iajc,ibjc->ab", t, t) - np.einsum("iajc,jbic->ab", t, t))
    return D_oo, D_vv


def mp2_density(Xo, Xv, Z):
    """(D_oo, D_vv) for the THC amplitudes of Eq.23 (Eqs.49-50 l.387-391 are Eqs.47-48 with Eq.23 inserted)."""
    return density_from_amplitudes(dense.expand_t(Xo, Xv, Z))


# ---- single elements, for shapes whose dense t (o^2 v^2 doubles) does not fit ----------------------------------------------
def _t_fixed_i(Xo, Xv, Z, i):
    """t[a, k, b] = t_ik^ab for one occupied index i (Eq.23)."""
    return np.einsum("aP,PQ,kQ,bQ->akb", Xv * Xo[i], Z, Xo, Xv, optimize=True)


def _t_fixed_a(Xo, Xv, Z, a):
    """t[i, j, c] = t_ij^ac for one virtual index a (Eq.23)."""
    return np.einsum("iP,PQ,jQ,cQ->ijc", Xo * Xv[a], Z, Xo, Xv, optimize=True)


def density_oo_element(Xo, Xv, Z, i, j):
    """D_ij of Eq.47 alone: -2 sum_kab t_ik^ab (2 t_jk^ab - t_jk^ba)."""
    ti, tj = _t_fixed_i(Xo, Xv, Z, i), _t_fixed_i(Xo, Xv, Z, j)
    return -2.0 * (2.0 * np.sum(ti * tj) - np.einsum("akb,bka->", ti, tj))


def density_vv_element(Xo, Xv, Z, a, b):
    """D_ab of Eq.48 alone: 2 sum_ijc t_ij^ac (2 t_ij^bc - t_ji^bc)."""
    ta, tb = _t_fixed_a(Xo, Xv, Z, a), _t_fixed_a(Xo, Xv, Z, b)
    return 2.0 * (2.0 * np.sum(ta * tb) - np.einsum("ijc,jic->", ta, tb))
