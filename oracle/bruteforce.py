"""T0 determinant-space brute force -- TEST INFRASTRUCTURE, not a product path.

Evaluates the closed-shell CCSD doubles residual and correlation energy at t1 = 0
from second quantisation alone -- no coupled-cluster working equation is used:

    T2    = 1/2 sum_ijab t_ij^ab E_ai E_bj,   E_ai = sum_sigma a+_{a sigma} a_{i sigma}
    psi   = (1 + T2 + T2^2 / 2) |Phi0>        (higher powers cannot reach a double through a two-body H)
    Omega_ij^ab = <D| H |psi> - t_ij^ab <Phi0| H |psi>,   D = E^alpha_ai E^beta_bj |Phi0>
                = <D| exp(-T2) H exp(T2) |Phi0>          (Eq.6 l.82 before projection)
    E_corr      = <Phi0| H |psi> - <Phi0| H |Phi0>       (Eq.2 l.65 with Lambda = 0)

    H = sum_pq h_pq a+_p a_q + 1/2 sum_pqrs <pq|rs> a+_p a+_q a_s a_r     (spin orbitals)
    <pq|rs> = (pr|qs) delta(spin p, spin r) delta(spin q, spin s)
    h = diag(eps) - sum_i [2 (pq|ii) - (pi|iq)]   so that the Fock matrix is diag(eps)
        (t1 = 0, canonical orbitals: reading R1/R8 of DESIGN.md)

Determinants are Python-int bit strings over 2(o+v) spin orbitals (index 2*P + spin);
operators act with explicit fermion signs.  Usable for (o, v) up to about (3, 3).

The bra <D| with one alpha and one beta excitation has <D|H|Phi0> = (ia|jb) and
<D|T2|Phi0> = t_ij^ab, i.e. it is the bra in which the paper's Omega (leading
term "(ai|bj)" with coefficient 1, Eq.29 l.224) is written.
"""
from __future__ import annotations

import itertools
import numpy as np


def _ann(det, p):
    """a_p |det> -> (sign, det') or None."""
    if not (det >> p) & 1:
        return None
    sign = -1 if bin(det & ((1 << p) - 1)).count("1") & 1 else 1
    return sign, det & ~(1 << p)


def _cre(det, p):
    """a+_p |det> -> (sign, det') or None."""
    if (det >> p) & 1:
        return None
    sign = -1 if bin(det & ((1 << p) - 1)).count("1") & 1 else 1
    return sign, det | (1 << p)


def _apply_string(det, ops):
    """Apply a product of operators given right-to-left as [(kind, p), ...] (first entry acts first)."""
    sign = 1
    for kind, p in ops:
        r = _ann(det, p) if kind == "a" else _cre(det, p)
        if r is None:
            return None
        sign *= r[0]
        det = r[1]
    return sign, det


def _vec_add(vec, det, val):
    if val != 0.0:
        vec[det] = vec.get(det, 0.0) + val


def apply_T2(vec, t, o, v):
    """(1/2 sum_ijab t[i,a,j,b] E_ai E_bj) |vec>   (vec: dict det -> coefficient)."""
    out = {}
    for det, c in vec.items():
        for i in range(o):
            for a in range(v):
                for j in range(o):
                    for b in range(v):
                        amp = 0.5 * t[i, a, j, b]
                        if amp == 0.0:
                            continue
                        for s in (0, 1):
                            for s2 in (0, 1):
                                # E_ai E_bj: E_bj acts first
                                r = _apply_string(det, [("a", 2 * j + s2), ("c", 2 * (o + b) + s2),
                                                        ("a", 2 * i + s), ("c", 2 * (o + a) + s)])
                                if r is not None:
                                    _vec_add(out, r[1], c * amp * r[0])
    return out


def apply_H(vec, h, eri, n):
    """H |vec> with spatial h[p,q] and chemists' ERIs eri[p,q,r,s] = (pq|rs)."""
    nso = 2 * n
    out = {}
    for det, c in vec.items():
        occ = [p for p in range(nso) if (det >> p) & 1]
        # one-body: sum_pq h_pq a+_p a_q  (spin conserving)
        for q in occ:
            r1 = _ann(det, q)
            for P in range(n):
                p = 2 * P + (q & 1)
                hv = h[P, q >> 1]
                if hv == 0.0:
                    continue
                r2 = _cre(r1[1], p)
                if r2 is not None:
                    _vec_add(out, r2[1], c * hv * r1[0] * r2[0])
        # two-body: 1/2 sum_pqrs <pq|rs> a+_p a+_q a_s a_r ; a_r acts first, then a_s
        for r in occ:
            rr = _ann(det, r)
            for s in occ:
                if s == r:
                    continue
                rs = _ann(rr[1], s)
                sgn_rs = rr[0] * rs[0]
                for Q in range(n):
                    q = 2 * Q + (s & 1)          # spin(q) = spin(s)
                    rq = _cre(rs[1], q)
                    if rq is None:
                        continue
                    for P in range(n):
                        p = 2 * P + (r & 1)      # spin(p) = spin(r)
                        val = eri[P, r >> 1, Q, s >> 1]    # <pq|rs> = (pr|qs)
                        if val == 0.0:
                            continue
                        rp = _cre(rq[1], p)
                        if rp is not None:
                            _vec_add(out, rp[1], 0.5 * c * val * sgn_rs * rq[0] * rp[0])
    return out


def full_eri(B_oo, B_ov, B_vv):
    """(pq|rs) over all o+v spatial orbitals from the Cholesky blocks (vo block = ov^T, t1 = 0)."""
    NL, o, v = B_ov.shape
    n = o + v
    B = np.zeros((NL, n, n))
    B[:, :o, :o] = B_oo
    B[:, :o, o:] = B_ov
    B[:, o:, :o] = B_ov.transpose(0, 2, 1)
    B[:, o:, o:] = B_vv
    return np.einsum("Lpq,Lrs->pqrs", B, B)


def omega_bruteforce(t, eri, eps, o, v):
    """Return (Omega[i,a,j,b], E_corr) by explicit action on determinants."""
    n = o + v
    h = np.diag(np.asarray(eps, dtype=float)).copy()
    for i in range(o):
        h -= 2.0 * eri[:, :, i, i] - eri[:, i, i, :]
    phi0 = (1 << (2 * o)) - 1
    psi0 = {phi0: 1.0}
    psi1 = apply_T2(psi0, t, o, v)
    psi2 = apply_T2(psi1, t, o, v)
    psi = dict(psi0)
    for d, c in psi1.items():
        _vec_add(psi, d, c)
    for d, c in psi2.items():
        _vec_add(psi, d, 0.5 * c)
    hpsi = apply_H(psi, h, eri, n)
    e_ref = apply_H(psi0, h, eri, n).get(phi0, 0.0)
    e_tot = hpsi.get(phi0, 0.0)
    omega = np.zeros((o, v, o, v))
    for i, a, j, b in itertools.product(range(o), range(v), range(o), range(v)):
        # D = a+_{a alpha} a_{i alpha} a+_{b beta} a_{j beta} |Phi0>   (beta pair acts first)
        r = _apply_string(phi0, [("a", 2 * j + 1), ("c", 2 * (o + b) + 1),
                                 ("a", 2 * i), ("c", 2 * (o + a))])
        sign, det = r
        omega[i, a, j, b] = sign * hpsi.get(det, 0.0) - t[i, a, j, b] * e_tot
    return omega, e_tot - e_ref


# ---- with singles: <mu| exp(-T) H exp(T) |Phi0>, T = T1 + T2 (no CC formula, no T1-dressing identity) --------------------
def apply_T1(vec, t1, o, v):
    """(sum_ia t1[i,a] E_ai) |vec>."""
    out = {}
    for det, c in vec.items():
        for i in range(o):
            for a in range(v):
                if t1[i, a] == 0.0:
                    continue
                for s in (0, 1):
                    r = _apply_string(det, [("a", 2 * i + s), ("c", 2 * (o + a) + s)])
                    if r is not None:
                        _vec_add(out, r[1], c * t1[i, a] * r[0])
    return out


def _exp_T(vec, t1, t, o, v, sign):
    """exp(sign * (T1 + T2)) |vec> by its (terminating) power series."""
    out, term, n = dict(vec), dict(vec), 0
    while term:
        n += 1
        nxt = apply_T1(term, t1, o, v)
        for d, c in apply_T2(term, t, o, v).items():
            _vec_add(nxt, d, c)
        term = {d: sign * c / n for d, c in nxt.items() if c != 0.0}
        for d, c in term.items():
            _vec_add(out, d, c)
        if n > 4 * (o + v):
            raise RuntimeError("series did not terminate")
    return out


def residuals_bruteforce_t1(t1, t, eri, eps, o, v):
    """(sigma[i,a], Omega[i,a,j,b]) = <mu| exp(-T) H exp(T) |Phi0> for the alpha single and the alpha-beta double
    excitation bras; h is fixed by the BARE Fock matrix being diag(eps), `eri` are the bare (pq|rs)."""
    n = o + v
    h = np.diag(np.asarray(eps, dtype=float)).copy()
    for i in range(o):
        h -= 2.0 * eri[:, :, i, i] - eri[:, i, i, :]
    phi0 = (1 << (2 * o)) - 1
    psi = _exp_T({phi0: 1.0}, t1, t, o, v, +1.0)
    r = _exp_T(apply_H(psi, h, eri, n), t1, t, o, v, -1.0)
    sigma = np.zeros((o, v))
    for i, a in itertools.product(range(o), range(v)):
        sg, det = _apply_string(phi0, [("a", 2 * i), ("c", 2 * (o + a))])
        sigma[i, a] = sg * r.get(det, 0.0)
    omega = np.zeros((o, v, o, v))
    for i, a, j, b in itertools.product(range(o), range(v), range(o), range(v)):
        sg, det = _apply_string(phi0, [("a", 2 * j + 1), ("c", 2 * (o + b) + 1), ("a", 2 * i), ("c", 2 * (o + a))])
        omega[i, a, j, b] = sg * r.get(det, 0.0)
    return sigma, omega
