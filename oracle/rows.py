"""T2 semi-dense oracle: sampled rows R[P, :] of every term -- TEST INFRASTRUCTURE, not a product path.

For shapes where the dense oracle (dense.py) cannot hold t_ijab or the 4-index ERIs (BASELINE configs 2-4) this file
evaluates, for a sampled amplitude-grid point P and each term of Omega separately,

    r^P_jb  = sum_ia U[ia,P] Omega_iajb ,        R[P, Q] = sum_jb r^P_jb U[jb,Q] ,       U[ia,P] = Xo[i,P] Xv[a,P]

(north_star projection; Eq.6 l.82 with U -> Xo.Xv, Eq.23 l.193).  Omega is the same sum of dense equations as
in dense.py (Eqs.28, 29, 31, 32+33, 35 corrected, 41 in Alg.9's symmetric form; readings R1-R7 of DESIGN.md) with the
row vector w_ia = U[ia,P] contracted in first.  Nothing of the factorised algorithms is used:

  * the amplitudes enter only through the literal definition t[i,a,j,b] = sum_PQ Xo_iP Xv_aP Z_PQ Xo_jQ Xv_bQ, written
    out as one einsum per contraction (`_t`), never through the Gram matrices o_PQ, v_PQ or the C^L, D^L, E, F, G, H
    intermediates of Algs.1-9;
  * the Cholesky ERIs enter as sum_L B^L (x) B^L applied one L-block at a time (Eq.24 l.199), the THC ERIs as
    sum_IJ (Yo Yv)_I V_IJ (Yo Yv)_J (Eq.17 l.141).

Cost per row: NL applications of t to an o x v matrix for s1/s3 (~5e12 flop at config 3), matrix-vector
work for s2/s7/s9, o v NX^2 for s6; xi_oo / xi_vv (Eqs.39-40) are full matrices and are computed once per input set.

Pinned by tests/test_oracle_rows.py against dense.py (itself pinned by the determinant-space brute force) on small and
ragged shapes, per term.
"""
from __future__ import annotations

import numpy as np

TERMS = ("s1", "s2", "s3", "s6", "s7", "s9")


class RowOracle:
    """Holds one input set; `row(P)` returns {term: R[P, :]}.

    B_vv may be an array [NL, v, v] or a callable bvv(L0, L1) -> [L1-L0, v, v] (paper-scale inputs are only ever
    materialised in L-blocks).  `lblock` bounds the temporaries of the L loop.
    """

    def __init__(self, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, lblock=16):
        self.Xo, self.Xv, self.Z, self.B_ov, self.B_oo, self.B_vv = Xo, Xv, Z, B_ov, B_oo, B_vv
        self.o, self.NP = Xo.shape
        self.v = Xv.shape[0]
        self.NL = B_ov.shape[0]
        self.Yo, self.Yv, self.V = Y[: self.o], Y[self.o:], V
        self.eps_o, self.eps_v = eps[: self.o], eps[self.o:]
        self.lblock = lblock
        self._xi = None

    # ---- the amplitudes, by their definition (Eq.23 l.193) ---------------------------------------------------------
    def _t(self, tidx, other, oidx, out):
        """sum over the shared letters of  t[tidx] * other[oidx]  ->  out, with t[i,a,j,b] = sum_PQ Xo_iP Xv_aP Z_PQ
        Xo_jQ Xv_bQ spelled out.  tidx is a 4-letter string (i, a, j, b positions); P, Q are reserved letters."""
        i, a, j, b = tidx
        spec = f"{i}P,{a}P,PQ,{j}Q,{b}Q,{oidx}->{out}"
        # the explicit memory limit only lets the path search form intermediates larger than its operands (e.g. [L,P,Q]);
        # the default limit would force a single 5-operand step of naive scaling
        return np.einsum(spec, self.Xo, self.Xv, self.Z, self.Xo, self.Xv, other, optimize=("optimal", 2 ** 34))

    def _u(self, x):
        """(u x)_kc = sum_ia (2 t_ik^ac - t_ik^ca) x_ia,  u[i,a,k,c] = 2 t[i,a,k,c] - t[i,c,k,a]."""
        return 2.0 * self._t("iakc", x, "ia", "kc") - self._t("icka", x, "ia", "kc")

    def _bvv(self, L0, L1):
        return self.B_vv(L0, L1) if callable(self.B_vv) else self.B_vv[L0:L1]

    def _lblocks(self):
        for L0 in range(0, self.NL, self.lblock):
            yield L0, min(self.NL, L0 + self.lblock)

    # ---- xi intermediates (Eqs.39-40 l.280-283; Cholesky ERIs) ---------------------------------------------------------
    def xi(self):
        """xi_oo[k,j] = sum_mde t_jm^de [2(me|kd) - (md|ke)];  xi_vv[b,c] = -sum_lmd t_lm^db [2(ld|mc) - (lc|md)]."""
        if self._xi is None:
            xi_oo = np.zeros((self.o, self.o))
            xi_vv = np.zeros((self.v, self.v))
            for L0, L1 in self._lblocks():
                B = self.B_ov[L0:L1]                                        # [l, m, e]
                # n[l,j,d] = sum_me (2 t[j,d,m,e] - t[j,e,m,d]) B^l_me
                n = 2.0 * self._t("jdme", B, "Lme", "Ljd") - self._t("jemd", B, "Lme", "Ljd")
                xi_oo += np.einsum("Lkd,Ljd->kj", B, n, optimize=True)      # (me|kd) -> B_me B_kd ; (md|ke) likewise
                xi_vv -= np.einsum("Lmb,Lmc->bc", n, B, optimize=True)
            self._xi = (xi_oo, xi_vv)
        return self._xi

    def xi_oo_column(self, j):
        """xi_oo[:, j] alone (Eq.39 l.280 with the index j fixed): for shapes where the full xi costs hours of CPU.
        n[L,d] = sum_me (2 t_jm^de - t_jm^ed) B^L_me,  xi_oo[k,j] = sum_Ld B^L_kd n[L,d]."""
        xo = self.Xo[j]
        col = np.zeros(self.o)
        lim = ("optimal", 2 ** 34)
        for L0, L1 in self._lblocks():
            B = self.B_ov[L0:L1]
            n = 2.0 * np.einsum("P,dP,PQ,mQ,eQ,Lme->Ld", xo, self.Xv, self.Z, self.Xo, self.Xv, B, optimize=lim) \
                - np.einsum("P,eP,PQ,mQ,dQ,Lme->Ld", xo, self.Xv, self.Z, self.Xo, self.Xv, B, optimize=lim)
            col += np.einsum("Lkd,Ld->k", B, n, optimize=True)
        return col

    def xi_vv_row(self, b):
        """xi_vv[b, :] alone (Eq.40 l.283 with the index b fixed):
        n[L,m] = sum_le (2 t_ml^be - t_ml^eb) B^L_le,  xi_vv[b,c] = -sum_Lm n[L,m] B^L_mc."""
        xv = self.Xv[b]
        row = np.zeros(self.v)
        lim = ("optimal", 2 ** 34)
        for L0, L1 in self._lblocks():
            B = self.B_ov[L0:L1]
            n = 2.0 * np.einsum("mP,P,PQ,lQ,eQ,Lle->Lm", self.Xo, xv, self.Z, self.Xo, self.Xv, B, optimize=lim) \
                - np.einsum("mP,eP,PQ,lQ,Q,Lle->Lm", self.Xo, self.Xv, self.Z, self.Xo, xv, B, optimize=lim)
            row -= np.einsum("Lm,Lmc->c", n, B, optimize=True)
        return row

    # ---- one row -----------------------------------------------------------------------------------------------------
    def row(self, P, terms=TERMS):
        """{term: R[P, :]} for the requested terms (each the projection of that term's Omega alone)."""
        w = np.outer(self.Xo[:, P], self.Xv[:, P])            # w_ia = U[ia, P]
        out = {}
        for k in terms:
            r = getattr(self, "_row_" + k)(w, P)              # r^P_jb
            out[k] = np.einsum("jb,jQ,bQ->Q", r, self.Xo, self.Xv, optimize=True)
        return out

    def _row_s2(self, w, P):
        """Eq.29 l.224:  (ia|jb) + sum_kc u_ik^ac (jb|kc) + sum_kc u_jk^bc (ia|kc)."""
        x = self._u(w)                                        # x_kc = sum_ia w_ia u_ik^ac
        g = np.zeros_like(w)                                  # g_kc = sum_ia w_ia (ia|kc)
        r = np.zeros_like(w)
        for L0, L1 in self._lblocks():
            B = self.B_ov[L0:L1]
            alpha = np.einsum("ia,Lia->L", w, B, optimize=True)
            beta = np.einsum("kc,Lkc->L", x, B, optimize=True)
            gl = np.einsum("L,Ljb->jb", alpha, B, optimize=True)
            g += gl
            r += gl + np.einsum("L,Ljb->jb", beta, B, optimize=True)
        return r + self._u(g)                                 # third term: sum_kc u_jk^bc g_kc

    def _row_s1(self, w, P):
        """Eq.28 l.217:  sum_cd t_ij^cd (ac|bd) + sum_kl t_kl^ab (ki|lj) - sum_lc t_il^cb (ac|lj) - sum_kd t_kj^ad (ki|bd)."""
        r = np.zeros_like(w)
        for L0, L1 in self._lblocks():
            Boo, Bvv = self.B_oo[L0:L1], self._bvv(L0, L1)
            Wv = np.einsum("ia,Lac->Lic", w, Bvv, optimize=True)       # sum_a w_ia B^L_ac
            Wo = np.einsum("Lki,ia->Lka", Boo, w, optimize=True)       # sum_i B^L_ki w_ia
            y1 = self._t("icjd", Wv, "Lic", "Ljd")                     # sum_ic t_ij^cd Wv_ic
            y2 = self._t("kalb", Wo, "Lka", "Llb")                     # sum_ka t_kl^ab Wo_ka
            r += np.einsum("Ljd,Lbd->jb", y1, Bvv, optimize=True)      # term 1
            r += np.einsum("Llj,Llb->jb", Boo, y2, optimize=True)      # term 2
            r -= np.einsum("Llj,Llb->jb", Boo, y1, optimize=True)      # term 3: sum_l (lj| sum_ic t_il^cb Wv_ic
            r -= np.einsum("Ljd,Lbd->jb", y2, Bvv, optimize=True)      # term 4: sum_d |bd) sum_ka t_kj^ad Wo_ka
        return r

    def _row_s3(self, w, P):
        """Eq.31 l.235:  - sum_kc [ t_ik^ac (kj|bc) + t_jk^bc (ki|ac) ]."""
        x = self._t("iakc", w, "ia", "kc")                    # sum_ia w_ia t_ik^ac
        r = np.zeros_like(w)
        q = np.zeros_like(w)                                  # q_kc = sum_ia w_ia (ki|ac)
        for L0, L1 in self._lblocks():
            Boo, Bvv = self.B_oo[L0:L1], self._bvv(L0, L1)
            r -= np.einsum("Lkj,kc,Lbc->jb", Boo, x, Bvv, optimize=True)
            q += np.einsum("Lki,ia,Lac->kc", Boo, w, Bvv, optimize=True)
        return r - self._t("jbkc", q, "kc", "jb")

    def _row_s9(self, w, P):
        """Eq.41 l.290 in Alg.9's symmetric form, F' = diag(eps) + xi:
        sum_c t_ij^ac F'_bc + sum_c t_ij^cb F'_ac - sum_k t_ik^ab F'_kj - sum_k t_kj^ab F'_ki."""
        xi_oo, xi_vv = self.xi()
        Foo = np.diag(self.eps_o) + xi_oo                     # F'[k, j]
        Fvv = np.diag(self.eps_v) + xi_vv                     # F'[b, c]
        x = self._t("iajc", w, "ia", "jc")                    # sum_ia w_ia t_ij^ac
        r = np.einsum("jc,bc->jb", x, Fvv, optimize=True)
        r += self._t("icjb", np.einsum("ia,ac->ic", w, Fvv, optimize=True), "ic", "jb")
        r -= np.einsum("kb,kj->jb", self._t("iakb", w, "ia", "kb"), Foo, optimize=True)
        r -= self._t("kajb", np.einsum("ia,ki->ka", w, Foo, optimize=True), "ka", "jb")
        return r

    # ---- THC-ERI terms ---------------------------------------------------------------------------------------------------
    def _thc_direct(self, x):
        """y_ld = sum_kc x_kc <kc|ld>   (Eq.17 l.141)."""
        s = np.einsum("kc,kI,cI->I", x, self.Yo, self.Yv, optimize=True)
        return np.einsum("I,IJ,lJ,dJ->ld", s, self.V, self.Yo, self.Yv, optimize=True)

    def _thc_exchange(self, x):
        """y_ld = sum_kc x_kc <kd|lc>."""
        return np.einsum("kc,kI,dI,IJ,lJ,cJ->ld", x, self.Yo, self.Yv, self.V, self.Yo, self.Yv,
                         optimize=("optimal", 2 ** 34))

    def _row_s7(self, w, P):
        """Eq.35 l.261 corrected (R2, R3): 1/2 sum_klcd [ u_ik^ac (2<kc|ld> - <kd|lc>) u_jl^bd + t_ik^ca <kd|lc> t_jl^db ]."""
        x1 = self._u(w)                                       # sum_ia w_ia u_ik^ac
        y1 = 2.0 * self._thc_direct(x1) - self._thc_exchange(x1)
        x2 = self._t("icka", w, "ia", "kc")                   # sum_ia w_ia t_ik^ca
        y2 = self._thc_exchange(x2)
        return 0.5 * (self._u(y1) + self._t("jdlb", y2, "ld", "jb"))       # t_jl^db = t[j,d,l,b]

    def _row_s6(self, w, P, ichunk=64):
        """Eqs.32+33 l.244-247:  sum_klcd t_ij^cd t_kl^ab <kc|ld> + sum_klcd t_ik^cb t_lj^ad <lc|kd>.
        With w_ia = Xo_iP Xv_aP:  theta[c,j,d] = sum_i Xo_iP t_ij^cd,  tau[k,l,b] = sum_a Xv_aP t_kl^ab, then
        r_jb = sum_klcd theta[c,j,d] <kc|ld> tau[k,l,b]  +  sum_klcd theta[c,k,b] <lc|kd> tau[l,j,d],
        the THC ERIs expanded over (I, J) in chunks of I."""
        xo, xv = self.Xo[:, P], self.Xv[:, P]
        theta = self._t("icjd", xo, "i", "cjd")
        tau = self._t("kalb", xv, "a", "klb")
        r = np.zeros_like(w)
        NX = self.V.shape[0]
        for I0 in range(0, NX, ichunk):
            I1 = min(NX, I0 + ichunk)
            Yo_c, Yv_c, V_c = self.Yo[:, I0:I1], self.Yv[:, I0:I1], self.V[I0:I1]
            # Eq.32: <kc|ld> = sum_IJ Yo_kI Yv_cI V_IJ Yo_lJ Yv_dJ
            th = np.einsum("cjd,cI,dJ->jIJ", theta, Yv_c, self.Yv, optimize=True)
            ta = np.einsum("klb,kI,lJ->bIJ", tau, Yo_c, self.Yo, optimize=True)
            r += (V_c[None] * th).reshape(self.o, -1) @ ta.reshape(self.v, -1).T          # sum_IJ V_IJ th[j,I,J] ta[b,I,J]
            # Eq.33: <lc|kd> = sum_IJ Yo_lI Yv_cI V_IJ Yo_kJ Yv_dJ
            ph = np.einsum("ckb,cI,kJ->bIJ", theta, Yv_c, self.Yo, optimize=True)
            ps = np.einsum("ljd,lI,dJ->jIJ", tau, Yo_c, self.Yv, optimize=True)
            r += (V_c[None] * ps).reshape(self.o, -1) @ ph.reshape(self.v, -1).T          # sum_IJ V_IJ ps[j,I,J] ph[b,I,J]
        return r

    # ---- energy (reading R7): E = sum_ijab (2 t_ij^ab - t_ij^ba)(ia|jb), Cholesky ERIs, in extended precision ------------
    def energy(self):
        """sum_L vec(B^L_ov)^T (2t - t^x) vec(B^L_ov), the L-sum accumulated in long double."""
        acc = np.longdouble(0.0)
        for L0, L1 in self._lblocks():
            B = self.B_ov[L0:L1]
            n = 2.0 * self._t("iajb", B, "Ljb", "Lia") - self._t("ibja", B, "Ljb", "Lia")
            acc += np.sum(np.einsum("Lia,Lia->L", n, B, optimize=True).astype(np.longdouble))
        return float(acc)
