"""Closed forms, special cases and invariants that pin oracle/dense.py."""
import copy

import numpy as np
import pytest

from conftest import small_inputs, oracle_eval
from oracle import dense

TERMS = dense.TERMS


def _inp(seed=21, dims=(3, 4, 6, 5, 7)):
    return small_inputs(*dims, seed=seed)


def test_each_term_and_total_symmetric():
    res = oracle_eval(_inp())
    for k in TERMS + ("R",):
        assert np.abs(res[k] - res[k].T).max() <= 1e-13 * max(1.0, np.abs(res[k]).max()), k


def test_permutational_symmetries_of_oracle_tensors():
    x = _inp()
    res = oracle_eval(x)
    t = res["t"]
    assert np.abs(t - t.transpose(2, 3, 0, 1)).max() < 1e-14          # t_ij^ab = t_ji^ba (l.178)
    cd = dense.cd_eris(x.B_oo, x.B_ov, x.B_vv)
    assert np.abs(cd["ovov"] - cd["ovov"].transpose(2, 3, 0, 1)).max() < 1e-14
    assert np.abs(cd["vvvv"] - cd["vvvv"].transpose(1, 0, 2, 3)).max() < 1e-14   # pq/qp
    assert np.abs(cd["oooo"] - cd["oooo"].transpose(0, 1, 3, 2)).max() < 1e-14
    for k in TERMS:
        om = res["omega"][k]
        assert np.abs(om - om.transpose(2, 3, 0, 1)).max() <= 1e-13 * np.abs(om).max(), k  # ia<->jb


def test_zero_amplitudes_give_bare_integrals():
    """Z = 0  =>  R_PQ = sum_L a^L_P a^L_Q with a^L_P = sum_ia Xo_iP Xv_aP B^L_ia; E = 0."""
    x = _inp()
    x.Z = np.zeros_like(x.Z)
    res = oracle_eval(x)
    A = np.einsum("iP,aP,Lia->PL", x.Xo, x.Xv, x.B_ov)
    assert np.abs(res["R"] - A @ A.T).max() < 1e-13
    for k in ("s1", "s3", "s6", "s7", "s9"):
        assert np.abs(res[k]).max() == 0.0
    assert res["E"] == 0.0


def test_zero_amplitudes_and_zero_integrals_give_zero():
    """north_star: R = 0 when Z = 0 and the ERIs are zero."""
    x = _inp()
    x.Z = np.zeros_like(x.Z)
    x.B_oo, x.B_ov, x.B_vv = (np.zeros_like(a) for a in (x.B_oo, x.B_ov, x.B_vv))
    res = oracle_eval(x)
    assert np.abs(res["R"]).max() == 0.0


def test_no_integrals_closed_form_orbital_energy_differences():
    """B = 0, V = 0  =>  Omega_ijab = (eps_a + eps_b - eps_i - eps_j) t_ij^ab  (reading R8)."""
    x = _inp()
    o = x.o
    x.B_oo, x.B_ov, x.B_vv = (np.zeros_like(a) for a in (x.B_oo, x.B_ov, x.B_vv))
    x.V = np.zeros_like(x.V)
    res = oracle_eval(x)
    eo, ev = x.eps[:o], x.eps[o:]
    D = ev[None, :, None, None] + ev[None, None, None, :] - eo[:, None, None, None] - eo[None, None, :, None]
    U = np.einsum("iP,aP->iaP", x.Xo, x.Xv)
    ref = np.einsum("iaP,iajb,jbQ->PQ", U, D * res["t"], U)
    assert np.abs(res["R"] - ref).max() <= 1e-13 * np.abs(ref).max()
    assert np.abs(res["s9"] - ref).max() <= 1e-13 * np.abs(ref).max()


def test_polynomial_structure_in_Z():
    """R(sZ) = R0 + s R1 + s^2 R2 exactly;  R2 = s6 + s7 + s9|eps=0,  R0 = A A^T."""
    x = _inp()
    r = {}
    for s in (0.0, 1.0, -1.0, 2.0):
        y = copy.deepcopy(x)
        y.Z = s * x.Z
        r[s] = oracle_eval(y)["R"]
    R0 = r[0.0]
    R2 = 0.5 * (r[1.0] + r[-1.0]) - R0
    R1 = 0.5 * (r[1.0] - r[-1.0])
    assert np.abs(r[2.0] - (R0 + 2 * R1 + 4 * R2)).max() <= 1e-12 * np.abs(r[2.0]).max()
    y = copy.deepcopy(x)
    y.eps = np.zeros_like(x.eps)
    q = oracle_eval(y)
    assert np.abs(R2 - (q["s6"] + q["s7"] + q["s9"])).max() <= 1e-12 * np.abs(R2).max()


def test_bilinear_in_B():
    x = _inp()
    r0 = oracle_eval(x)
    y = copy.deepcopy(x)
    y.B_oo, y.B_ov, y.B_vv = 2 * x.B_oo, 2 * x.B_ov, 2 * x.B_vv
    r1 = oracle_eval(y)
    for k in ("s1", "s2", "s3"):
        assert np.abs(r1[k] - 4 * r0[k]).max() <= 1e-12 * np.abs(r1[k]).max()
    for k in ("s6", "s7"):
        assert np.abs(r1[k] - r0[k]).max() == 0.0
    assert r1["E"] == pytest.approx(4 * r0["E"], rel=1e-13)


def test_cholesky_rotation_invariance():
    """B^L -> sum_M Q_LM B^M with Q orthogonal leaves every (pq|rs), hence R and E, unchanged."""
    x = _inp()
    r0 = oracle_eval(x)
    rng = np.random.default_rng(0)
    Q, _ = np.linalg.qr(rng.standard_normal((x.NL, x.NL)))
    y = copy.deepcopy(x)
    y.B_oo = np.einsum("LM,Mpq->Lpq", Q, x.B_oo)
    y.B_ov = np.einsum("LM,Mpq->Lpq", Q, x.B_ov)
    y.B_vv = np.einsum("LM,Mpq->Lpq", Q, x.B_vv)
    r1 = oracle_eval(y)
    for k in TERMS + ("R",):
        assert np.abs(r1[k] - r0[k]).max() <= 1e-12 * max(1.0, np.abs(r0[k]).max()), k
    assert r1["E"] == pytest.approx(r0["E"], abs=1e-12)


def test_grid_gauge_invariance():
    """Xo_P -> alpha_P Xo_P, Xv_P -> Xv_P / alpha_P leaves U^P_ia and R unchanged; same for (Y, V)."""
    x = _inp()
    r0 = oracle_eval(x)
    rng = np.random.default_rng(1)
    al = rng.uniform(0.5, 2.0, x.NP)
    be = rng.uniform(0.5, 2.0, x.NX)
    y = copy.deepcopy(x)
    y.Xo = x.Xo * al[None, :]
    y.Xv = x.Xv / al[None, :]
    y.Y = x.Y.copy()
    y.Y[: x.o] = x.Y[: x.o] * be[None, :]
    y.V = x.V / (be[:, None] * be[None, :])
    r1 = oracle_eval(y)
    for k in TERMS + ("R",):
        assert np.abs(r1[k] - r0[k]).max() <= 1e-12 * max(1.0, np.abs(r0[k]).max()), k


def test_zero_padding_invariance():
    x = _inp()
    r0 = oracle_eval(x)
    y = copy.deepcopy(x)
    pad = 3
    y.Xo = np.pad(x.Xo, ((0, 0), (0, pad)))
    y.Xv = np.pad(x.Xv, ((0, 0), (0, pad)))
    y.Z = np.pad(x.Z, ((0, pad), (0, pad)))
    y.B_oo = np.pad(x.B_oo, ((0, 2), (0, 0), (0, 0)))
    y.B_ov = np.pad(x.B_ov, ((0, 2), (0, 0), (0, 0)))
    y.B_vv = np.pad(x.B_vv, ((0, 2), (0, 0), (0, 0)))
    y.Y = np.pad(x.Y, ((0, 0), (0, 4)))
    y.V = np.pad(x.V, ((0, 4), (0, 4)))
    r1 = oracle_eval(y)
    NP = x.NP
    assert np.abs(r1["R"][:NP, :NP] - r0["R"]).max() <= 1e-13 * np.abs(r0["R"]).max()
    assert np.abs(r1["R"][NP:, :]).max() == 0.0 and np.abs(r1["R"][:, NP:]).max() == 0.0


def test_direct_ring_limit():
    """Coulomb-only ring (dRPA-like) limit pins the factor 1/2 and the '2's of Eq.35 / Eq.29 independently
    of T0: with t_ij^ba dropped (u -> 2t) and exchange integrals dropped, in the composite-index matrix
    form  Omega = K + 2 K T + 2 T K + 4 T K T  for T = t[(ia),(jb)], K = (ia|jb) = <ia|jb>."""
    x = _inp()
    t = dense.expand_t(x.Xo, x.Xv, x.Z)
    ovov = np.einsum("Lia,Ljb->iajb", x.B_ov, x.B_ov)
    n = x.o * x.v
    Tm, Km = t.reshape(n, n), ovov.reshape(n, n)
    ref = Km + 2 * Km @ Tm + 2 * Tm @ Km + 4 * Tm @ Km @ Tm
    # the same pieces as coded in the oracle's formulas: Eq.29 with u -> 2t, Eq.35 first bracket with
    # u -> 2t, w -> 2<.|.>, prefactor 1/2
    u = 2.0 * t
    s2 = ovov + np.einsum("iakc,jbkc->iajb", u, ovov) + np.einsum("jbkc,iakc->iajb", u, ovov)
    s7 = 0.5 * np.einsum("iakc,kcld,jbld->iajb", u, 2.0 * ovov, u, optimize=True)
    assert np.abs((s2 + s7).reshape(n, n) - ref).max() <= 1e-12 * np.abs(ref).max()


def test_energy_closed_form_factorised():
    """E = sum_L [ 2 a^T Z a - sum_PQ Z_PQ E^L_PQ E^L_QP ],  a^L, E^L from B_ov."""
    x = _inp()
    res = oracle_eval(x)
    e = 0.0
    for L in range(x.NL):
        EL = x.Xo.T @ x.B_ov[L] @ x.Xv          # E^L[P,Q] = sum_ia Xo_iP B_ia Xv_aQ
        a = np.diag(EL)
        e += 2 * a @ x.Z @ a - np.sum(x.Z * EL * EL.T)
    assert res["E"] == pytest.approx(e, rel=1e-12)
