"""Pins of oracle/rr.py (rank-reduced working variables, Eqs.9-14, 22)."""
import numpy as np

from conftest import small_inputs, oracle_eval
from oracle import rr, dense


def _problem(NR=4, seed=31):
    x = small_inputs(3, 4, 6, 7, 9, seed=seed, zmul=30.0)
    rng = np.random.default_rng(seed)
    tau = rng.standard_normal((NR, x.NP))
    T = rng.standard_normal((NR, NR))
    return x, tau, 0.5 * (T + T.T)


def test_orthogonalised_projectors_are_semi_unitary():
    """Eq.12 l.112: sum_ia U~^P_ia U~^Q_ia = delta_PQ after tau~ = S^{-1/2} tau (Eqs.10-13)."""
    x, tau, _ = _problem()
    U = rr.projectors(x.Xo, x.Xv, rr.symmetric_orthogonalizer(x.Xo, x.Xv, tau))
    G = np.einsum("iaP,iaQ->PQ", U, U)
    assert np.abs(G - np.eye(tau.shape[0])).max() < 1e-12
    U0 = rr.projectors(x.Xo, x.Xv, tau)                     # the raw CP factors are NOT semi-unitary
    assert np.abs(np.einsum("iaP,iaQ->PQ", U0, U0) - np.eye(tau.shape[0])).max() > 1e-2


def test_identity_tau_reduces_to_the_grid_residual():
    """tau~ = 1 (NR = NP): U~ = Xo.Xv, T = Z, so R^RR is the oracle of record's R and E its E."""
    x, _, _ = _problem()
    ref = oracle_eval(x)
    got = rr.rr_residual_and_energy(x.Xo, x.Xv, np.eye(x.NP), x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
    assert np.abs(got["R_rr"] - ref["R"]).max() <= 1e-12 * np.abs(ref["R"]).max()
    assert abs(got["E"] - ref["E"]) <= 1e-12 * max(1.0, abs(ref["E"]))


def test_amplitudes_and_projection_follow_eq22_and_eq6_by_loops():
    """t_ij^ab = sum_PQ U~^P_ia T^PQ U~^Q_jb and R^RR_PQ = sum U~^P_ia Omega_ijab U~^Q_jb written as literal loops
    (a transposed tau or a swapped index would show), and the THC-basis core Z = tau~^T T tau~ reproduces t (Eq.22)."""
    x, tau, T = _problem(NR=3)
    tau = rr.symmetric_orthogonalizer(x.Xo, x.Xv, tau)
    got = rr.rr_residual_and_energy(x.Xo, x.Xv, tau, T, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
    o, v, NR, NP = x.o, x.v, 3, x.NP
    U = np.zeros((o, v, NR))
    for i in range(o):
        for a in range(v):
            for P in range(NR):
                U[i, a, P] = sum(x.Xo[i, W] * x.Xv[a, W] * tau[P, W] for W in range(NP))
    t = np.zeros((o, v, o, v))
    for P in range(NR):
        for Q in range(NR):
            t += T[P, Q] * np.multiply.outer(U[:, :, P], U[:, :, Q])
    assert np.abs(t - got["t"]).max() < 1e-13 * np.abs(t).max()
    Z = tau.T @ T @ tau
    assert np.abs(dense.expand_t(x.Xo, x.Xv, Z) - t).max() < 1e-12 * np.abs(t).max()
    ref = dense.residual_and_energy(x.Xo, x.Xv, Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
    omega = sum(ref["omega"][k] for k in dense.TERMS)
    R = np.zeros((NR, NR))
    for P in range(NR):
        for Q in range(NR):
            R[P, Q] = np.sum(U[:, :, P][:, :, None, None] * omega * U[:, :, Q][None, None, :, :])
    assert np.abs(R - got["R_rr"]).max() <= 1e-12 * np.abs(R).max()
    assert np.abs(got["R_rr"] - got["R_rr"].T).max() <= 1e-12 * np.abs(R).max()
