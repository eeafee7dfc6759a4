"""Pins of oracle/t1.py (T1-dressed singles and doubles residuals, Eqs.24-29, 31, 38, 41, 42)."""
import numpy as np
import pytest

from conftest import small_inputs, oracle_eval
from oracle import dense, t1 as t1o, bruteforce


def _t1(o, v, seed, scale=0.3):
    return scale * np.random.default_rng(seed).standard_normal((o, v))


@pytest.mark.parametrize("o,v,seed", [(2, 3, 11), (2, 2, 13), (3, 3, 12)])
def test_t1_residuals_equal_determinant_bruteforce(o, v, seed):
    """<mu| exp(-T1-T2) H exp(T1+T2) |0> from bit-string determinants: singles and doubles, O(1) amplitudes."""
    x = small_inputs(o, v, 7, 5, 9, seed=seed)
    tt = _t1(o, v, seed)
    res = t1o.residual_and_energy(x.Xo, x.Xv, x.Z, tt, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps, thc_from_cd=True)
    eri = bruteforce.full_eri(x.B_oo, x.B_ov, x.B_vv)
    sig_bf, om_bf = bruteforce.residuals_bruteforce_t1(tt, res["t"], eri, x.eps, o, v)
    om = sum(res["omega"][k] for k in dense.TERMS)
    assert np.abs(om - om_bf).max() <= 1e-11 * np.abs(om_bf).max()
    assert np.abs(res["sigma"] - sig_bf).max() <= 1e-11 * np.abs(sig_bf).max()
    # the pin must bite: t1 changes both residuals at O(1), and both singles groups matter
    ref0 = oracle_eval(x, thc_from_cd=True)
    assert np.abs(om - sum(ref0["omega"][k] for k in dense.TERMS)).max() > 1e-2 * np.abs(om).max()
    assert min(np.abs(res["sigma_G_H"]).max(), np.abs(res["sigma_I_J"]).max()) > 1e-3 * np.abs(sig_bf).max()


def test_t1_zero_reduces_to_the_oracle_of_record():
    x = small_inputs(3, 4, 6, 5, 7, seed=5)
    ref = oracle_eval(x)
    res = t1o.residual_and_energy(x.Xo, x.Xv, x.Z, np.zeros((3, 4)), x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
    for k in dense.TERMS + ("R", "xi_oo", "xi_vv"):
        assert np.abs(res[k] - ref[k]).max() <= 1e-13 * max(1.0, np.abs(ref[k]).max()), k
    assert np.abs(res["F"] - np.diag(x.eps)).max() < 1e-12       # canonical orbitals: F = diag(eps)


def test_dressing_identities():
    """B^_ia = B_ia (l.145: ovov-type integrals untouched); bra-ket symmetry only (l.211); the blockwise formulas that
    the CUDA path uses for B^_oo, B^_vv, B^_vo."""
    x = small_inputs(3, 4, 6, 5, 7, seed=6)
    o, v = 3, 4
    tt = _t1(o, v, 2)
    B = t1o.full_B(x.B_oo, x.B_ov, x.B_vv)
    Bh = t1o.dress(B, tt)
    assert np.abs(Bh[:, :o, o:] - x.B_ov).max() < 1e-14
    assert np.abs(Bh[:, :o, :o] - (x.B_oo + np.einsum("Lka,ja->Lkj", x.B_ov, tt))).max() < 1e-13
    assert np.abs(Bh[:, o:, o:] - (x.B_vv - np.einsum("ia,Lib->Lab", tt, x.B_ov))).max() < 1e-13
    S = np.einsum("Lab,ib->Lai", Bh[:, o:, o:], tt)
    assert np.abs(Bh[:, o:, :o] - (x.B_ov.transpose(0, 2, 1) - np.einsum("ja,Lji->Lai", tt, x.B_oo) + S)).max() < 1e-13
    g = np.einsum("Lpq,Lrs->pqrs", Bh, Bh)
    assert np.abs(g - g.transpose(2, 3, 0, 1)).max() < 1e-13
    assert np.abs(g - g.transpose(1, 0, 2, 3)).max() > 1e-3
